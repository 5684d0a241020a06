// NEXT-3, second half — sub-sample alignment of the detectors' SNR series (reading X7, DESIGN.md
// §11c): around every candidate the window z[k - H .. k + H] of each detector is resampled R
// times finer with the cubic Lagrange interpolator through the four neighbouring samples; the
// coherent search (k_sky) then runs unchanged on those windows with a delay table built at R
// times the sampling rate ("Time offsets of SNRs from different detectors", taken
// on a finer grid).
//
//   out[I][s][u] = z_I(row_s, k_s - H + u / R),  u = 0 .. 2 R H;   the candidate sits at u = R H
//   u = R q + r:  r = 0  the sample itself (bit copy)
//                 r > 0  w_r[0] z[b-1] + w_r[1] z[b] + w_r[2] z[b+1] + w_r[3] z[b+2],  b = k_s - H + q,
//                        float32, one multiply then three fused multiply-adds per component
// One CTA per (slot, detector), threads stride over the output samples (coalesced stores, reads of 2 H + 3
// consecutive ring samples served by L1 across the R phases; one 64-bit modulo per thread, then wraps).
// HBM-bound: 8 (2 H + 3) B read + 8 (2 R H + 2) B written per (slot, detector).
#include <cstring>

#include "spiir_internal.cuh"

namespace spiir {

constexpr int kUpThreads = 128;
constexpr int kUpMaxFactor = 16;

struct UpParams {
  const float2* z; int64_t det_stride, row_stride, ring_len, k_newest, n_rows;
  const spiir_trigger* trig; int32_t n_slots, n_det;
  int32_t S1;                                        // rows per slot: 1 (foreground) or the number of slides
  int32_t slides;                                    // 1: row (slot, s) holds the windows of slide s + 1
  int64_t step; int32_t mult[SPIIR_MAX_DET];
  int32_t R, H, Lw; int64_t Lp;
  float4 w[kUpMaxFactor];
  float2* out; spiir_trigger* trig_out;
};

// Centre of detector I's window for row (slot, si): the candidate's sample, moved s step mult[I] earlier in the
// detectors other than the trigger detector for slide s = si + 1; ok = every detector's window and
// its interpolation margin lie in the view.
__device__ __forceinline__ bool up_row(const UpParams& P, const spiir_trigger& t, int si, int64_t* centre) {
  const int64_t k_old = P.k_newest - P.ring_len + 1 > 0 ? P.k_newest - P.ring_len + 1 : 0;
  bool ok = t.valid && t.tmpl >= 0 && t.tmpl < P.n_rows && t.det >= 0 && t.det < P.n_det;
  for (int I = 0; I < P.n_det; ++I) {
    const int64_t c = t.k - ((P.slides && I != t.det) ? (int64_t)(si + 1) * P.step * P.mult[I] : 0);
    centre[I] = c;
    ok = ok && c - P.H - 1 >= k_old && c + P.H + 1 <= P.k_newest;
  }
  return ok;
}

// the re-addressed candidates (one thread per row)
__global__ void __launch_bounds__(kUpThreads) k_upsample_trig(const __grid_constant__ UpParams P) {
  const int w = blockIdx.x * kUpThreads + threadIdx.x;
  if (w >= P.n_slots * P.S1) return;
  const int s = w / P.S1, si = w - s * P.S1;
  const spiir_trigger t = P.trig[s];
  int64_t centre[SPIIR_MAX_DET];
  const bool ok = up_row(P, t, si, centre);
  spiir_trigger o = t;
  o.valid = ok ? 1 : 0; o.tmpl = w; o.k = (int64_t)P.R * P.H;
  if (!t.valid) { o.det = 0; o.z_re = o.z_im = o.snr = 0.f; }
  o._pad = 0; o._pad2 = 0.f;
  P.trig_out[w] = o;
}

// the windows: one CTA per (slot, detector), threads stride over the output samples (coalesced stores; the
// 2 H + 3 ring samples a window reads are consecutive and stay in L1 across the R phases).  One 64-bit
// modulo per thread places the window in the ring; after that a sample's neighbours are conditional wraps.
__global__ void __launch_bounds__(kUpThreads) k_upsample(const __grid_constant__ UpParams P) {
  const int w = blockIdx.x, I = blockIdx.y;
  const int s = w / P.S1, si = w - s * P.S1;
  const spiir_trigger t = P.trig[s];
  int64_t centre[SPIIR_MAX_DET];
  const bool ok = up_row(P, t, si, centre);
  float2* out = P.out + ((size_t)I * P.n_slots * P.S1 + w) * P.Lp;
  if (!ok) {
    for (int u = threadIdx.x; u < P.Lp; u += kUpThreads) out[u] = make_float2(0.f, 0.f);
    return;
  }
  const float2* zr = P.z + (size_t)I * P.det_stride + (size_t)t.tmpl * P.row_stride;
  const int64_t L = P.ring_len;
  const int64_t i0 = (centre[I] - P.H) % L;              // centre - H >= 1 here
  auto wrap = [L](int64_t i) { return i >= L ? i - L : (i < 0 ? i + L : i); };
  for (int u = threadIdx.x; u < P.Lp; u += kUpThreads) {
    float2 v = make_float2(0.f, 0.f);
    if (u < P.Lw) {
      const int q = u / P.R, r = u - q * P.R;
      // q <= 2 H: if the window is longer than the ring the validity test above has already failed
      const int64_t i = wrap(i0 + q);
      if (r == 0) {
        v = zr[i];
      } else {
        const float4 w = P.w[r];
        const float2 z0 = zr[wrap(i - 1)], z1 = zr[i], z2 = zr[wrap(i + 1)], z3 = zr[wrap(wrap(i + 1) + 1)];
        v.x = __fmaf_rn(w.w, z3.x, __fmaf_rn(w.z, z2.x, __fmaf_rn(w.y, z1.x, __fmul_rn(w.x, z0.x))));
        v.y = __fmaf_rn(w.w, z3.y, __fmaf_rn(w.z, z2.y, __fmaf_rn(w.y, z1.y, __fmul_rn(w.x, z0.y))));
      }
    }
    out[u] = v;
  }
}

}  // namespace spiir

using namespace spiir;

extern "C" {

int spiir_snr_upsample_elems(int32_t n_det, int32_t n_slots, int32_t factor, int32_t half_width, size_t* elems) {
  SPIIR_REQUIRE(elems != nullptr, "elems is NULL");
  SPIIR_REQUIRE(n_det >= 1 && n_det <= SPIIR_MAX_DET && n_slots >= 0, "bad n_det / n_slots");
  SPIIR_REQUIRE(factor >= 1 && factor <= kUpMaxFactor, "factor %d out of range 1..%d", factor, kUpMaxFactor);
  SPIIR_REQUIRE(half_width >= 1 && half_width <= (1 << 20), "half_width out of range");
  const size_t Lp = ((size_t)2 * factor * half_width + 1 + 1) & ~(size_t)1;
  *elems = (size_t)n_det * n_slots * Lp;
  return SPIIR_OK;
}

static int upsample_run(const spiir_snr_view* view, int32_t n_det, const spiir_trigger* dev_trig, int32_t n_slots,
                        int32_t n_slides, int64_t step, const int32_t* mult, int32_t factor, int32_t half_width,
                        spiir_c32* dev_out, spiir_trigger* dev_trig_out, spiir_snr_view* out_view, void* stream) {
  size_t elems = 0;
  int rc = spiir_snr_upsample_elems(n_det, n_slots, factor, half_width, &elems);
  if (rc) return rc;
  SPIIR_REQUIRE(dev_trig && dev_out && dev_trig_out && out_view, "a pointer is NULL");
  if (int rcv = check_snr_view(view)) return rcv;
  SPIIR_REQUIRE(view->k_newest >= 0, "view: k_newest < 0");
  SPIIR_REQUIRE(((uintptr_t)dev_out & 15) == 0, "dev_out must be 16-byte aligned");
  if (int rcs = check_slides(n_slides, step, mult, n_det)) return rcs;
  const int S1 = n_slides > 0 ? n_slides : 1;
  SPIIR_REQUIRE((long long)n_slots * S1 <= 0x7fffffffLL, "too many rows");
  UpParams P;
  memset(&P, 0, sizeof(P));
  P.z = (const float2*)view->dev_z;
  P.det_stride = view->det_stride; P.row_stride = view->row_stride;
  P.ring_len = view->ring_len; P.k_newest = view->k_newest; P.n_rows = view->n_rows;
  P.trig = dev_trig; P.n_slots = n_slots; P.n_det = n_det;
  P.S1 = S1; P.slides = n_slides > 0 ? 1 : 0; P.step = step;
  for (int I = 0; I < SPIIR_MAX_DET; ++I) P.mult[I] = (n_slides > 0 && I < n_det) ? mult[I] : 0;
  P.R = factor; P.H = half_width; P.Lw = 2 * factor * half_width + 1;
  P.Lp = ((int64_t)P.Lw + 1) & ~(int64_t)1;
  for (int r = 0; r < kUpMaxFactor; ++r) {
    // cubic through nodes -1, 0, 1, 2 evaluated at mu = r / R, in float64, rounded once
    const double m = r < factor ? (double)r / factor : 0.0;
    P.w[r] = make_float4((float)(-m * (m - 1.0) * (m - 2.0) / 6.0), (float)((m + 1.0) * (m - 1.0) * (m - 2.0) / 2.0),
                         (float)(-(m + 1.0) * m * (m - 2.0) / 2.0), (float)((m + 1.0) * m * (m - 1.0) / 6.0));
  }
  P.out = (float2*)dev_out; P.trig_out = dev_trig_out;
  const long long n_rows = (long long)n_slots * S1;
  out_view->dev_z = dev_out;
  out_view->det_stride = n_rows * P.Lp;
  out_view->row_stride = P.Lp;
  out_view->ring_len = P.Lp;
  out_view->k_newest = P.Lw - 1;
  out_view->n_rows = n_rows;
  if (n_rows == 0) return SPIIR_OK;
  k_upsample_trig<<<(unsigned)((n_rows + kUpThreads - 1) / kUpThreads), kUpThreads, 0, (cudaStream_t)stream>>>(P);
  k_upsample<<<dim3((unsigned)n_rows, (unsigned)n_det), kUpThreads, 0, (cudaStream_t)stream>>>(P);
  count_launch(2);
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

int spiir_snr_upsample_windows(const spiir_snr_view* view, int32_t n_det, const spiir_trigger* dev_trig,
                               int32_t n_slots, int32_t factor, int32_t half_width, spiir_c32* dev_out,
                               spiir_trigger* dev_trig_out, spiir_snr_view* out_view, void* stream) {
  return upsample_run(view, n_det, dev_trig, n_slots, 0, 0, nullptr, factor, half_width, dev_out, dev_trig_out, out_view, stream);
}

int spiir_snr_upsample_windows_slides(const spiir_snr_view* view, int32_t n_det, const spiir_trigger* dev_trig,
                                      int32_t n_slots, int32_t n_slides, int64_t step_samples,
                                      const int32_t* host_slide_mult, int32_t factor, int32_t half_width,
                                      spiir_c32* dev_out, spiir_trigger* dev_trig_out, spiir_snr_view* out_view,
                                      void* stream) {
  SPIIR_REQUIRE(n_slides >= 1, "n_slides must be >= 1");
  return upsample_run(view, n_det, dev_trig, n_slots, n_slides, step_samples, host_slide_mult, factor, half_width,
                      dev_out, dev_trig_out, out_view, stream);
}

}  // extern "C"
