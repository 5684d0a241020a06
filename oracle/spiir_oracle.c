/*
 * spiir_oracle.c — float64 CPU ORACLE for the SPIIR hot path (arXiv 2011.06787).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call it.
 * It shares no code, header, table or constant with the CUDA path under
 * paper_2011_06787_b200/.  It is deliberately plain: every function follows the
 * paper's definition step by step, sequential in time, in double / complex
 * double, with no blocking, scans, fusion or re-association.  OpenMP is used
 * only to run independent templates / triggers on different cores.
 *
 * Steps (readings A1-A27 / M1-M9 listed in DESIGN.md):
 *   O1 decimator       BASELINE.json config 2 (32-tap half-band FIR); not in PAPER.md
 *   O2 recursion       PAPER.md:129 (Eq. 8): y_l[k] = a_l y_l[k-1] + b_l x[k-d_l]
 *   O3 sum / combine   PAPER.md:122 ("summation of responses from all IIR filters")
 *   O4 peaks
 *   O6 coherent / null PAPER.md:147-157 (Eq. 9, 10), PAPER.md:483-495 (Eq. 28-30)
 *   O7 time slides
 *   O8 xi^2 (NEXT-1)   PAPER.md:177-188 (Eq. 11, 12)
 * (O5, the look-up table build, is in oracle/sky.py because it uses numpy's SVD.)
 *
 * Pins (tests/test_oracle_pins.py): P1 impulse response, P2 brute-force
 * convolution, P4 linearity/shift, P5 scipy lfilter/upfirdn, P6 periodic
 * shift-invariance, P8 B=1 special case, P9 brute-force peaks, P10-P13, P16.
 * PARITY UNPINNED (no external truth, only the stated reading): the multirate
 * combination M4-M6 beyond its scipy.upfirdn restatement, the time-slide
 * pattern A16.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define EXPORT __attribute__((visibility("default")))

/* ---------------------------------------------------------------- O1 ---- */
/* x_{b+1}[m] = sum_{j<ntaps} g[j] x_b[2m+1-j],  x_b[n<0] = 0   (reading M3) */
EXPORT void spiir_oracle_decimate(const double* x, int64_t n, const double* g, int ntaps, double* y)
{
    for (int64_t m = 0; m < n / 2; ++m) {
        double acc = 0.0;
        for (int j = 0; j < ntaps; ++j) {
            int64_t i = 2 * m + 1 - j;
            if (i >= 0) acc += g[j] * x[i];
        }
        y[m] = acc;
    }
}

/* ------------------------------------------------------------ O2 + O3 --- */
/* Band sum of one template in one band: s[m] = sum_l y_l[m] in filter order,
 * y_l[m] = a_l y_l[m-1] + b_l x[m-d_l], y_l[-1] = 0, x[<0] = 0 (A1, A6).
 * a, b are the float32 coefficients (re, im interleaved) promoted to double (A5). */
EXPORT void spiir_oracle_band_sum(const double* x, int64_t n, int64_t nf,
                                  const float* a, const float* b, const int32_t* d,
                                  double* s /* [n][2], overwritten */)
{
    memset(s, 0, sizeof(double) * 2 * (size_t)n);
    for (int64_t l = 0; l < nf; ++l) {
        const double ar = a[2 * l], ai = a[2 * l + 1];
        const double br = b[2 * l], bi = b[2 * l + 1];
        double yr = 0.0, yi = 0.0;
        for (int64_t m = 0; m < n; ++m) {
            const int64_t i = m - d[l];
            const double u = (i >= 0) ? x[i] : 0.0;
            const double nr = ar * yr - ai * yi + br * u;
            const double ni = ar * yi + ai * yr + bi * u;
            yr = nr; yi = ni;
            s[2 * m] += yr;
            s[2 * m + 1] += yi;
        }
    }
}

/* acc_b[m] = s_b[m] + sum_{j<ntaps} h[j] v[m-j],  v[i] = acc_{b+1}[i/2] for even
 * i >= 0, else 0 (zero stuffing, readings M4).  h already holds the factor 2. */
EXPORT void spiir_oracle_interp_add(const double* acc_next /* [n/2][2] */, int64_t n,
                                    const double* h, int ntaps,
                                    const double* s /* [n][2] or NULL */, double* acc /* [n][2] */)
{
    for (int64_t m = 0; m < n; ++m) {
        double re = s ? s[2 * m] : 0.0, im = s ? s[2 * m + 1] : 0.0;
        for (int j = 0; j < ntaps; ++j) {
            const int64_t i = m - j;
            if (i >= 0 && (i % 2) == 0) {
                re += h[j] * acc_next[2 * (i / 2)];
                im += h[j] * acc_next[2 * (i / 2) + 1];
            }
        }
        acc[2 * m] = re; acc[2 * m + 1] = im;
    }
}

/* Whole bank, one shot over the full stream, for a list of selected templates.
 * z[det][sel][m] at the output band's rate.  out_band must be 0 or 1 (M5):
 *   out_band == 0:  z = acc_0
 *   out_band == 1:  z[m] = acc_1[m] + s_0[2m+1]
 * Returns 0, or -1 on bad arguments. */
EXPORT int spiir_oracle_bank(int n_det, int64_t n0, const float* strain /* [n_det][n0] */,
                             int n_bands, int out_band,
                             int64_t n_sel, const int64_t* sel, const int64_t* tmpl_offset,
                             const float* a, const float* b, const int32_t* delay, const uint8_t* band,
                             const float* dec_taps, const float* int_taps, int ntaps,
                             double* z /* [n_det][n_sel][n0 >> out_band][2] */)
{
    if (n_bands < 1 || n_bands > 8 || out_band < 0 || out_band > 1 || out_band >= n_bands) return -1;
    if (n0 % ((int64_t)1 << (n_bands - 1))) return -1;
    const int64_t n_out = n0 >> out_band;
    double g[64], h[64];
    for (int j = 0; j < ntaps; ++j) { g[j] = dec_taps ? dec_taps[j] : 0.0; h[j] = int_taps ? int_taps[j] : 0.0; }

    /* O1: the band inputs of every detector */
    double** xb = (double**)calloc((size_t)n_det * n_bands, sizeof(double*));
    for (int D = 0; D < n_det; ++D) {
        double* x0 = (double*)malloc(sizeof(double) * (size_t)n0);
        for (int64_t i = 0; i < n0; ++i) x0[i] = strain[(size_t)D * n0 + i];
        xb[D * n_bands] = x0;
        for (int bnd = 1; bnd < n_bands; ++bnd) {
            const int64_t nprev = n0 >> (bnd - 1);
            xb[D * n_bands + bnd] = (double*)malloc(sizeof(double) * (size_t)(nprev / 2));
            spiir_oracle_decimate(xb[D * n_bands + bnd - 1], nprev, g, ntaps, xb[D * n_bands + bnd]);
        }
    }

    #pragma omp parallel for schedule(dynamic, 1) collapse(2)
    for (int D = 0; D < n_det; ++D) {
        for (int64_t si = 0; si < n_sel; ++si) {
            const int64_t t = sel[si];
            const int64_t f0 = tmpl_offset[t], f1 = tmpl_offset[t + 1];
            const int64_t nf = f1 - f0;
            float* ta = (float*)malloc(sizeof(float) * 2 * (size_t)(nf + 1));
            float* tb = (float*)malloc(sizeof(float) * 2 * (size_t)(nf + 1));
            int32_t* td = (int32_t*)malloc(sizeof(int32_t) * (size_t)(nf + 1));
            double* sb[8]; double* acc = NULL;
            /* O2 + O3 band sums, filters taken in index order within each band */
            for (int bnd = 0; bnd < n_bands; ++bnd) {
                const int64_t nb = n0 >> bnd;
                int64_t c = 0;
                for (int64_t l = f0; l < f1; ++l)
                    if (band[l] == bnd) {
                        ta[2 * c] = a[2 * l]; ta[2 * c + 1] = a[2 * l + 1];
                        tb[2 * c] = b[2 * l]; tb[2 * c + 1] = b[2 * l + 1];
                        td[c] = delay[l]; ++c;
                    }
                sb[bnd] = (double*)malloc(sizeof(double) * 2 * (size_t)nb);
                spiir_oracle_band_sum(xb[D * n_bands + bnd], nb, c, ta, tb, td, sb[bnd]);
            }
            /* O3 cascade: acc_{B-1} = s_{B-1}; acc_b = s_b + up2(acc_{b+1}) down to out_band */
            acc = sb[n_bands - 1];
            for (int bnd = n_bands - 2; bnd >= out_band; --bnd) {
                const int64_t nb = n0 >> bnd;
                double* nacc = (double*)malloc(sizeof(double) * 2 * (size_t)nb);
                spiir_oracle_interp_add(acc, nb, h, ntaps, sb[bnd], nacc);
                free(acc);
                free(sb[bnd]);
                acc = nacc;
            }
            double* zo = z + 2 * ((size_t)D * n_sel + si) * (size_t)n_out;
            if (out_band == 0) {
                memcpy(zo, acc, sizeof(double) * 2 * (size_t)n_out);
            } else {                                          /* M5 */
                for (int64_t m = 0; m < n_out; ++m) {
                    zo[2 * m]     = acc[2 * m]     + sb[0][2 * (2 * m + 1)];
                    zo[2 * m + 1] = acc[2 * m + 1] + sb[0][2 * (2 * m + 1) + 1];
                }
                free(sb[0]);
            }
            free(acc); free(ta); free(tb); free(td);
        }
    }
    for (int i = 0; i < n_det * n_bands; ++i) free(xb[i]);
    free(xb);
    return 0;
}

/* ---------------------------------------------------------------- O4 ---- */
/* |z|^2 either in double (z double) or decided in float32 exactly as
 * fl(fl(re*re) + fl(im*im)) when z is float32 (the kernel's precision). */
static double mag2_at(const void* z, int is_f32, int64_t idx)
{
    if (is_f32) {
        const float* p = (const float*)z + 2 * idx;
        volatile float rr = p[0] * p[0];
        volatile float ii = p[1] * p[1];
        volatile float s = rr + ii;
        return (double)s;
    }
    const double* p = (const double*)z + 2 * idx;
    return p[0] * p[0] + p[1] * p[1];
}
static double thr2_of(double thr, int is_f32)
{
    if (is_f32) { volatile float t = (float)thr; volatile float t2 = t * t; return (double)t2; }
    return thr * thr;
}

/* mode 0: per row (= one template of one detector) arg-max over the n samples,
 * lowest index on exact ties; valid iff |z|^2 > thr^2 (strict, A11). */
EXPORT void spiir_oracle_peaks_mode0(int64_t n_rows, int64_t n, const void* z, int is_f32,
                                     double thr, int64_t* k_out, int32_t* valid)
{
    const double t2 = thr2_of(thr, is_f32);
    for (int64_t r = 0; r < n_rows; ++r) {
        int64_t best = 0; double bm = -1.0;
        for (int64_t k = 0; k < n; ++k) {
            const double m2 = mag2_at(z, is_f32, r * n + k);
            if (m2 > bm) { bm = m2; best = k; }
        }
        k_out[r] = best;
        valid[r] = (bm > t2) ? 1 : 0;
    }
}

/* mode 1 for one detector and one chunk: z[n_templates][n].
 * Per bank of bank_size consecutive templates: (i) at each sample the template
 * with the largest |z|^2 (lowest t on ties), kept iff > thr^2; (ii) per template
 * the kept sample with the largest |z|^2 (lowest k on ties). */
EXPORT void spiir_oracle_peaks_mode1(int64_t n_templates, int64_t n, int64_t bank_size,
                                     const void* z, int is_f32, double thr,
                                     int64_t* k_out, int32_t* valid)
{
    const double t2 = thr2_of(thr, is_f32);
    for (int64_t t = 0; t < n_templates; ++t) { valid[t] = 0; k_out[t] = 0; }
    double* best = (double*)malloc(sizeof(double) * (size_t)n_templates);
    for (int64_t t = 0; t < n_templates; ++t) best[t] = -1.0;
    for (int64_t t0 = 0; t0 < n_templates; t0 += bank_size) {
        const int64_t t1 = (t0 + bank_size < n_templates) ? t0 + bank_size : n_templates;
        for (int64_t k = 0; k < n; ++k) {
            int64_t ts = t0; double bm = -1.0;
            for (int64_t t = t0; t < t1; ++t) {
                const double m2 = mag2_at(z, is_f32, t * n + k);
                if (m2 > bm) { bm = m2; ts = t; }
            }
            if (bm > t2 && bm > best[ts]) { best[ts] = bm; k_out[ts] = k; valid[ts] = 1; }
        }
    }
    free(best);
}

/* ------------------------------------------------------------ O6 / O7 --- */
typedef struct {
    int n_det; int64_t n_pix;
    const float* u2; const int32_t* delay;
    const void* z; int z_is_f32;
    int64_t det_stride, row_stride, ring_len, k_newest;
} sky_ctx;

static int in_range(const sky_ctx* c, int64_t kk)
{
    int64_t lo = c->k_newest - c->ring_len + 1;
    if (lo < 0) lo = 0;
    return kk >= lo && kk <= c->k_newest;
}
static void z_at(const sky_ctx* c, int det, int64_t row, int64_t kk, double* re, double* im)
{
    const int64_t idx = det * c->det_stride + row * c->row_stride + (kk % c->ring_len);
    if (c->z_is_f32) { const float* p = (const float*)c->z + 2 * idx; *re = p[0]; *im = p[1]; }
    else             { const double* p = (const double*)c->z + 2 * idx; *re = p[0]; *im = p[1]; }
}

/* One evaluation of Eq. 9 / Eq. 10 at pixel p (reading A14: z is the column
 * vector, rho_c^2 = sum_{j=1,2} |sum_I U_Ij z_I|^2).  shift[I] is the extra
 * (time-slide) offset of detector I, 0 in the foreground.  Returns 0 when a
 * gather index leaves the valid range of the view. */
static int eval_pixel(const sky_ctx* c, int64_t row, int trig_det, int64_t k, const int64_t* shift,
                      int64_t p, double* coh2, double* tot2)
{
    double c0r = 0, c0i = 0, c1r = 0, c1i = 0, tot = 0;
    const int32_t* dl = c->delay + p * c->n_det;
    const float* u = c->u2 + p * c->n_det * 2;
    for (int I = 0; I < c->n_det; ++I) {
        const int64_t kk = k - shift[I] + (int64_t)dl[I] - (int64_t)dl[trig_det];   /* A18: differences at use */
        if (!in_range(c, kk)) return 0;
        double vr, vi;
        z_at(c, I, row, kk, &vr, &vi);
        c0r += (double)u[2 * I] * vr;     c0i += (double)u[2 * I] * vi;
        c1r += (double)u[2 * I + 1] * vr; c1i += (double)u[2 * I + 1] * vi;
        tot += vr * vr + vi * vi;
    }
    *coh2 = c0r * c0r + c0i * c0i + c1r * c1r + c1i * c1i;
    *tot2 = tot;
    return 1;
}

/* Foreground (n_slides == 0) or time-slide background (n_slides >= 1).
 * out[n_trig][S][3] = coh2, null2, tot2 at the arg-max pixel (lowest p on exact
 * ties), pix_out[n_trig][S]; S = max(1, n_slides); slide s = 1..n_slides is
 * stored at index s-1 and reads detector I at k - s*step*mult[I] + Delta (O7).
 * A (trigger, slide) for which ANY pixel's gather leaves the view, or an invalid
 * trigger slot, yields pix = -1 and zeros.  skymap (foreground only, may be
 * NULL): coh2 for every pixel. */
EXPORT int spiir_oracle_sky(int n_det, int64_t n_pix, const float* u2, const int32_t* delay,
                            const void* z, int z_is_f32, int64_t det_stride, int64_t row_stride,
                            int64_t ring_len, int64_t k_newest,
                            int64_t n_trig, const int32_t* trig_valid, const int32_t* trig_row,
                            const int32_t* trig_det, const int64_t* trig_k,
                            int n_slides, int64_t step, const int32_t* slide_mult,
                            double* out, int32_t* pix_out, double* skymap)
{
    if (n_det < 2 || n_det > 8) return -1;
    const sky_ctx c = { n_det, n_pix, u2, delay, z, z_is_f32, det_stride, row_stride, ring_len, k_newest };
    const int S = n_slides > 0 ? n_slides : 1;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t i = 0; i < n_trig; ++i) {
        for (int s = 0; s < S; ++s) {
            double* o = out + ((size_t)i * S + s) * 3;
            int32_t* po = pix_out + (size_t)i * S + s;
            o[0] = o[1] = o[2] = 0.0; *po = -1;
            if (!trig_valid[i]) continue;
            int64_t shift[8];
            for (int I = 0; I < n_det; ++I)
                shift[I] = (n_slides > 0 && I != trig_det[i]) ? (int64_t)(s + 1) * step * slide_mult[I] : 0;
            int ok = 1; int64_t best = -1; double bc = -1.0, bt = 0.0;
            for (int64_t p = 0; p < n_pix; ++p) {
                double coh2, tot2;
                if (!eval_pixel(&c, trig_row[i], trig_det[i], trig_k[i], shift, p, &coh2, &tot2)) { ok = 0; break; }
                if (skymap && n_slides == 0) skymap[(size_t)i * n_pix + p] = coh2;
                if (coh2 > bc) { bc = coh2; bt = tot2; best = p; }
            }
            if (!ok) {
                if (skymap && n_slides == 0)
                    for (int64_t p = 0; p < n_pix; ++p) skymap[(size_t)i * n_pix + p] = 0.0;
                continue;
            }
            o[0] = bc; o[2] = bt;
            o[1] = (bt - bc > 0.0) ? bt - bc : 0.0;            /* Eq. 10, clamped (A25) */
            *po = (int32_t)best;
        }
    }
    return 0;
}

/* A single evaluation (trigger, slide s >= 0 with 0 = foreground, pixel p):
 * res[3] = coh2, null2 (unclamped tot2 - coh2), tot2.  Returns 1 if in range. */
EXPORT int spiir_oracle_sky_eval(int n_det, int64_t n_pix, const float* u2, const int32_t* delay,
                                 const void* z, int z_is_f32, int64_t det_stride, int64_t row_stride,
                                 int64_t ring_len, int64_t k_newest,
                                 int32_t row, int32_t trig_det, int64_t k,
                                 int s, int64_t step, const int32_t* slide_mult, int64_t p, double* res)
{
    const sky_ctx c = { n_det, n_pix, u2, delay, z, z_is_f32, det_stride, row_stride, ring_len, k_newest };
    int64_t shift[8];
    for (int I = 0; I < n_det; ++I)
        shift[I] = (s > 0 && I != trig_det) ? (int64_t)s * step * slide_mult[I] : 0;
    double coh2, tot2;
    if (!eval_pixel(&c, row, trig_det, k, shift, p, &coh2, &tot2)) { res[0] = res[1] = res[2] = 0; return 0; }
    res[0] = coh2; res[1] = tot2 - coh2; res[2] = tot2;
    return 1;
}

/* ---------------------------------------------------------------- O8 ---- */
/* Signal-consistency statistic, PAPER.md:177-188 (Eq. 11, 12):
 *   xi_I^2 = sum_{j=-nj}^{nj} |z_I[c_I + j] - z_I[c_I] A[j]|^2 / sum_j (2 - 2 |A[j]|^2),
 *   xi_C^2 = (1/N_d) sum_I xi_I^2,
 * with A = acorr[row][j + nj] the template's normalised autocorrelation (A[0] = 1)
 * and c_I = k + delay[pix][I] - delay[pix][T] the sample of detector I aligned with
 * the trigger at the direction `pix` found by the coherent search (reading X1 in
 * DESIGN.md).  n_slides = 0: foreground, pix[n_trig]; n_slides >= 1: the same for the
 * time-slid companions of O7, pix[n_trig][n_slides].  out[n_trig][S][n_det + 2] =
 * xi_I^2 ..., xi_C^2, used (1/0).  A slot that is invalid, has pix < 0, or whose window
 * leaves the view in any detector gives zeros. */
EXPORT int spiir_oracle_xi2(int n_det, const int32_t* delay,
                            const void* z, int z_is_f32, int64_t det_stride, int64_t row_stride,
                            int64_t ring_len, int64_t k_newest,
                            int64_t n_trig, const int32_t* trig_valid, const int32_t* trig_row,
                            const int32_t* trig_det, const int64_t* trig_k, const int32_t* pix,
                            int n_slides, int64_t step, const int32_t* slide_mult,
                            const double* acorr, int nj, double* out)
{
    if (n_det < 1 || n_det > 8 || nj < 1) return -1;
    const sky_ctx c = { n_det, 0, NULL, delay, z, z_is_f32, det_stride, row_stride, ring_len, k_newest };
    const int W = 2 * nj + 1;
    const int S = n_slides > 0 ? n_slides : 1;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n_trig; ++i) {
        for (int s = 0; s < S; ++s) {
            double* o = out + ((size_t)i * S + s) * (n_det + 2);
            const int32_t px = pix[(size_t)i * S + s];
            for (int q = 0; q < n_det + 2; ++q) o[q] = 0.0;
            if (!trig_valid[i] || px < 0) continue;
            const int32_t* dl = delay + (size_t)px * n_det;
            const double* A = acorr + (size_t)trig_row[i] * W * 2;
            int64_t ci[8];
            int ok = 1;
            for (int I = 0; I < n_det; ++I) {
                /* time slide s+1 reads detector I != T at k - (s+1) step m_I + Delta (O7) */
                const int64_t shift = (n_slides > 0 && I != trig_det[i]) ? (int64_t)(s + 1) * step * slide_mult[I] : 0;
                ci[I] = trig_k[i] - shift + (int64_t)dl[I] - (int64_t)dl[trig_det[i]];
                if (!in_range(&c, ci[I] - nj) || !in_range(&c, ci[I] + nj)) ok = 0;
            }
            if (!ok) continue;
            double den = 0.0;
            for (int j = 0; j < W; ++j) den += 2.0 - 2.0 * (A[2 * j] * A[2 * j] + A[2 * j + 1] * A[2 * j + 1]);
            double mean = 0.0;
            for (int I = 0; I < n_det; ++I) {
                double z0r, z0i, num = 0.0;
                z_at(&c, I, trig_row[i], ci[I], &z0r, &z0i);
                for (int j = -nj; j <= nj; ++j) {
                    double zr, zi;
                    z_at(&c, I, trig_row[i], ci[I] + j, &zr, &zi);
                    const double ar = A[2 * (j + nj)], ai = A[2 * (j + nj) + 1];
                    const double er = zr - (z0r * ar - z0i * ai), ei = zi - (z0r * ai + z0i * ar);
                    num += er * er + ei * ei;
                }
                o[I] = den > 0.0 ? num / den : 0.0;
                mean += o[I];
            }
            o[n_det] = mean / n_det;
            o[n_det + 1] = 1.0;
        }
    }
    return 0;
}

/* Thread count for the timed runs of bench.py (the physical cores of the box); no arithmetic here. */
EXPORT void spiir_oracle_set_threads(int n)
{
    #ifdef _OPENMP
    if (n >= 1) omp_set_num_threads(n);
    #else
    (void)n;
    #endif
}

EXPORT int spiir_oracle_num_threads(void)
{
    int n = 1;
    #ifdef _OPENMP
    #pragma omp parallel
    {
        #pragma omp single
        n = omp_get_num_threads();
    }
    #endif
    return n;
}
