/*
 * spiir.h — C ABI of the B200-native SPIIR hot path (arXiv 2011.06787).
 *
 * Two stages, both hand-written CUDA for sm_100a behind this boundary:
 *   1. the SPIIR filter bank  — PAPER.md:122-131 (Sec. II B 1, "Eq. 8"):
 *        z_t[k] = sum_{l in t} y_l[k],  y_l[k] = a_l y_l[k-1] + b_l x[k - d_l]
 *      over (multirate) whitened strain, with all state carried across streaming
 *      chunks, plus the per-second candidate selection of PAPER.md:162-167;
 *   2. the coherent sky search — PAPER.md:147-157 (Eq. 9, 10)
 *      (HEALPix directions, look-up tables of U and time offsets) and its
 *      time-slide background.
 *
 * Conventions
 *   - Every function returns an int status: SPIIR_OK or a negative SPIIR_E* code;
 *     spiir_last_error() gives the text of the last failure on this thread.
 *   - Pointers named host_* are host memory, dev_* are device memory owned by the
 *     caller.  The library owns only the opaque handle and the workspace carve-up;
 *     it never frees caller memory and allocates nothing after spiir_bank_init.
 *   - All device work is enqueued on the caller's stream (passed as void*, a
 *     cudaStream_t); no call synchronises the device.  Outputs are valid once the
 *     stream has been synchronised by the caller.
 *   - Complex numbers are interleaved (re, im) float32.
 *   - Sample indices k are ABSOLUTE output-rate sample counts since the last
 *     spiir_bank_reset (int64).
 */
#ifndef SPIIR_H
#define SPIIR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPIIR_OK          0
#define SPIIR_EINVAL     -1   /* null pointer, bad size, bands not halving, delay > max_delay, ... */
#define SPIIR_ENOMEM     -2   /* workspace too small */
#define SPIIR_ECUDA      -3   /* CUDA runtime error (text in spiir_last_error) */
#define SPIIR_EOVERFLOW  -4   /* a fixed-size internal table would overflow */

#define SPIIR_MAX_BANDS   8
#define SPIIR_MAX_DET     4
#define SPIIR_FIR_TAPS   32

typedef struct spiir_bank spiir_bank;              /* opaque */
typedef struct { float re, im; } spiir_c32;

/* Description of a filter bank (all arrays host memory, copied at init).
 * Filters are stored template by template (CSR); within a template in any order.
 * A filter l is the triple (a, b, delay) of PAPER.md:122 — feedback coefficient
 * (paper a_0, north_star a1), feed-forward coefficient (paper b_1, north_star b0),
 * integer delay in samples of ITS OWN band — plus the index of its rate band. */
typedef struct {
  int32_t n_det;                         /* 1..SPIIR_MAX_DET; coefficients are shared by detectors      */
  int32_t n_templates;
  int32_t n_bands;                       /* 1..SPIIR_MAX_BANDS                                          */
  int32_t out_band;                      /* band whose rate is the output rate; must be 0 or 1          */
  int32_t band_rate_hz[SPIIR_MAX_BANDS]; /* strictly halving: rate[b+1] * 2 == rate[b]                  */
  int32_t max_delay[SPIIR_MAX_BANDS];    /* history depth per band, samples of that band                */
  int64_t n_filters;                     /* total                                                        */
  const int64_t*   host_tmpl_offset;     /* [n_templates+1] CSR into the filter arrays                  */
  const spiir_c32* host_a;               /* [n_filters] feedback                                        */
  const spiir_c32* host_b;               /* [n_filters] feed-forward                                    */
  const int32_t*   host_delay;           /* [n_filters] 0 <= delay <= max_delay[band]                   */
  const uint8_t*   host_band;            /* [n_filters]                                                 */
  const float*     host_fir_dec;         /* [32] decimation taps: x_{b+1}[m] = sum_j g[j] x_b[2m+1-j]   */
  const float*     host_fir_int;         /* [32] interpolation taps h (factor 2 included):
                                            acc_b[m] = s_b[m] + sum_j h[j] v[m-j], v = zero-stuffed acc_{b+1} */
  int32_t max_chunk_samples;             /* largest n_samples of one spiir_filter_chunk call (band 0)   */
  int32_t bank_size;                     /* templates per "template bank" for peak mode 1 */
  int64_t ring_len;                      /* SNR history kept per (detector, template), output samples;
                                            >= max_chunk_samples >> out_band                            */
} spiir_bank_desc;

/* Device bytes spiir_bank_init needs for this bank (coefficients, IIR state, delay
 * lines, FIR / interpolator histories, band-sum scratch, SNR ring, peak slots). */
int spiir_bank_workspace_bytes(const spiir_bank_desc* desc, size_t* bytes);

/* Plans the device layout, copies the coefficients, zeroes all carried state.
 * dev_workspace: 256-byte aligned device memory of at least the queried size; it
 * must stay alive until spiir_bank_free.  Errors: EINVAL, ENOMEM, ECUDA. */
int spiir_bank_init(spiir_bank** out, const spiir_bank_desc* desc,
                    void* dev_workspace, size_t bytes, void* stream);

/* Zeroes every carried state (IIR states, histories, ring, sample counter). */
int spiir_bank_reset(spiir_bank* bank, void* stream);

/* Releases the host-side handle (never the workspace). */
int spiir_bank_free(spiir_bank* bank);

/* One streaming chunk (H0-H3 of DESIGN.md): decimate the strain into the rate
 * bands, run every filter's recursion over the chunk with its state carried
 * from the previous call, sum per template, combine the bands up to the output
 * rate, append the SNR to the ring and track each template's maximum.
 *   dev_strain : [n_det][n_samples] float32 at band_rate_hz[0]
 *   n_samples  : multiple of 4 * 2^(n_bands-1), <= max_chunk_samples
 *   dev_snr_out: [n_det][n_templates][n_samples >> out_band] complex, or NULL (ring only)
 */
int spiir_filter_chunk(spiir_bank* bank, const float* dev_strain, int32_t n_samples,
                       spiir_c32* dev_snr_out, void* stream);

/* A single-detector candidate.  40 bytes. */
typedef struct {
  int32_t valid;      /* 1 if this slot holds a candidate                          */
  int32_t tmpl;       /* template index (row of the SNR view)                      */
  int32_t det;        /* detector the candidate was found in                       */
  int32_t _pad;
  int64_t k;          /* absolute output-rate sample index of the maximum          */
  float   z_re, z_im; /* complex SNR there                                         */
  float   snr;        /* |z|                                                       */
  float   _pad2;
} spiir_trigger;

/* Candidate selection over the LAST chunk (H4).
 *   mode 0: per (detector, template) the sample of largest |z|^2 (lowest k on exact
 *           ties); valid iff |z|^2 > thr^2 (strict; thr = 0 keeps every slot).
 *   mode 1: the paper's two-step rule per bank of desc.bank_size templates:
 *           at each sample keep the loudest template if above threshold, then per
 *           template keep its loudest kept sample.
 * |z|^2 is decided in float32 as fl(fl(re*re) + fl(im*im)).
 *   dev_trig : [n_det][n_templates] dense slots (deterministic order)
 *   dev_count: one int32, number of valid slots */
int spiir_peaks(spiir_bank* bank, float snr_threshold, int32_t mode,
                spiir_trigger* dev_trig, int32_t* dev_count, void* stream);

/* A window onto complex SNR series: z(det,row,k) = dev_z[det*det_stride +
 * row*row_stride + (k mod ring_len)] (strides in complex elements), defined for
 * 0 <= row < n_rows and max(0, k_newest - ring_len + 1) <= k <= k_newest.  A trigger
 * slot whose tmpl is not a row of the view is treated as an empty slot.  48 bytes.
 * The struct carries no size or version field: zero-initialise it and set EVERY field (n_rows is the newest one; a
 * view with n_rows outside 1..2^31-1, a NULL dev_z, ring_len < 1 or a negative stride is refused with SPIIR_EINVAL by
 * every call that takes a view). */
typedef struct {
  const spiir_c32* dev_z;
  int64_t det_stride, row_stride;
  int64_t ring_len, k_newest;
  int64_t n_rows;
} spiir_snr_view;

/* The bank's own SNR ring as a view (rows = templates). */
int spiir_bank_snr_view(const spiir_bank* bank, spiir_snr_view* view);

/* Host helper (float64 inside, not on the hot path) — the per-direction look-up
 * table of: HEALPix RING pixel centres of `nside`,
 * G+ / Gx of each detector at psi = 0, U2 = first two left
 * singular vectors of the sensitivity-weighted response G_sigma (Eq. 27,
 * PAPER.md:473), delay = rint(-(r_I . n)/c * fs_hz) per detector against the
 * geocentre (differences delay[p][I] - delay[p][T] are taken at use).
 *   host_det_pos_m [n_det][3] Earth-fixed metres; host_det_resp [n_det][3][3]
 *   response tensors (x x^T - y y^T)/2; host_sigma [n_det] sensitivity weights.
 *   Outputs: host_u2 [12 nside^2][n_det][2], host_delay [12 nside^2][n_det]. */
int spiir_sky_table_build(int32_t nside, int32_t n_det, const double* host_det_pos_m,
                          const double* host_det_resp, const double* host_sigma,
                          double gmst_rad, double fs_hz, float* host_u2, int32_t* host_delay);

/* NEXT-3 — "we sample U every half hour up to 24 hours and
 * refreshed every day ... Time offsets ... are sampled at the same interval
 * along with U.  The pipeline will calculate the coherent SNR using the U and
 * offset sample that are closest in the time to the triggering candidate."
 * Set i (0 <= i < n_sets) is spiir_sky_table_build at sidereal angle
 * gmst0_rad + 2 pi i interval_s / 86164.0905 (one turn per sidereal day).
 *   Outputs: host_u2 [n_sets][12 nside^2][n_det][2], host_delay
 *   [n_sets][12 nside^2][n_det]; other arguments as spiir_sky_table_build. */
int spiir_sky_table_set_build(int32_t nside, int32_t n_det, const double* host_det_pos_m,
                              const double* host_det_resp, const double* host_sigma,
                              double gmst0_rad, double interval_s, int32_t n_sets, double fs_hz,
                              float* host_u2, int32_t* host_delay);

/* Index of the set closest in time to t_s when set i holds time t0_s +
 * i interval_s: the earlier set on an exact tie; *index = -1 (and SPIIR_OK)
 * when t_s is further than interval_s / 2 from every set, i.e. the tables are
 * stale and must be rebuilt (the paper refreshes them daily).  Host arithmetic
 * in float64; no device work. */
int spiir_sky_table_nearest(double t_s, double t0_s, double interval_s, int32_t n_sets, int32_t* index);

/* NEXT-3, second half (reading X7 of DESIGN.md) — sub-sample
 * alignment.  The paper aligns the detectors' SNR series at integer samples
 * ("Time offsets of SNRs from different detectors"); this call
 * resamples, around every candidate, the window z[k - H .. k + H] of each
 * detector `factor` times finer with the cubic Lagrange interpolator through the
 * four neighbouring samples, so that coherent_sky_search can run unchanged on the
 * windows with a table built at factor * fs_hz:
 *   dev_out[I][s][u] = z_I(row_s, k_s - H + u / factor), u = 0 .. 2 factor H
 *   (row stride padded to an even number of elements; samples with u a multiple
 *   of factor are bit copies; the others are w0 z[b-1] + w1 z[b] + w2 z[b+1] +
 *   w3 z[b+2] in float32: one multiply, then three fused multiply-adds per
 *   component, weights formed in float64 and rounded once).
 *   dev_trig_out[s] = the candidate re-addressed to its window: tmpl = s,
 *   k = factor * H, det / z / snr kept; valid = 0 (and an all-zero window) when
 *   the slot is empty or k - H - 1 .. k + H + 1 is not inside the view.
 *   *out_view describes dev_out (rows = slots).  factor 1..16; H must cover the
 *   largest inter-detector delay in input samples.  (The search on the windows needs
 *   the factor-times wider delay windows of at least 32 candidates in shared memory:
 *   for H1-L1-V1 at 2048 Hz that holds up to factor 3, 4 when the trigger is not in
 *   V1; spiir_sky_plan_init reports a table that does not fit as EINVAL.)  dev_out: 16-byte aligned,
 *   spiir_snr_upsample_elems() complex elements, caller-owned.  Asynchronous on
 *   `stream`.  Errors: EINVAL, ECUDA. */
int spiir_snr_upsample_elems(int32_t n_det, int32_t n_slots, int32_t factor, int32_t half_width, size_t* elems);
int spiir_snr_upsample_windows(const spiir_snr_view* view, int32_t n_det, const spiir_trigger* dev_trig,
                               int32_t n_slots, int32_t factor, int32_t half_width, spiir_c32* dev_out,
                               spiir_trigger* dev_trig_out, spiir_snr_view* out_view, void* stream);

/* The same for the time-slide background, so that foreground and background are the SAME statistic when
 * the sub-sample alignment is on: row s * n_slides + (slide - 1) of dev_out holds, for detector I, the window around
 * k_s - slide * step_samples * host_slide_mult[I] (the trigger detector's window is not moved), resampled as above;
 * dev_trig_out [n_slots * n_slides] re-addresses the candidate to that row (valid = 0 and zero windows when ANY
 * detector's window or its one-sample interpolation margin leaves the view).  coherent_sky_search on *out_view with
 * these slots returns results laid out [n_slots][n_slides], as timeslide_background does.
 * dev_out: n_slides * spiir_snr_upsample_elems() complex elements. */
int spiir_snr_upsample_windows_slides(const spiir_snr_view* view, int32_t n_det, const spiir_trigger* dev_trig,
                                      int32_t n_slots, int32_t n_slides, int64_t step_samples,
                                      const int32_t* host_slide_mult, int32_t factor, int32_t half_width,
                                      spiir_c32* dev_out, spiir_trigger* dev_trig_out, spiir_snr_view* out_view,
                                      void* stream);

/* A look-up table prepared for the device (opaque).  The plan re-orders the
 * directions so that those sharing one tuple of inter-detector delays are
 * adjacent, and stores for each direction the projector U2 U2^T (Eq. 28,
 * rho_c^2 = z^H U I U^T z) next to its pixel index.  Results are
 * always reported with the caller's pixel numbering. */
typedef struct spiir_sky_plan spiir_sky_plan;

/* Device bytes a plan for (n_det, n_pix) with outputs for up to max_slots
 * trigger slots needs (table stream + compaction lists). */
int spiir_sky_plan_workspace_bytes(int32_t n_det, int32_t n_pix, int32_t max_slots, size_t* bytes);

/* host_u2 [n_pix][n_det][2] float32, host_delay [n_pix][n_det] int32 (any table,
 * e.g. from spiir_sky_table_build; copied).  dev_workspace: 256-byte aligned,
 * alive until spiir_sky_plan_free.  n_det 2..SPIIR_MAX_DET.  Synchronises the
 * stream once (setup, not hot path).  Errors: EINVAL, ENOMEM, ECUDA. */
int spiir_sky_plan_init(spiir_sky_plan** out, int32_t n_det, int32_t n_pix, int32_t max_slots,
                        const float* host_u2, const int32_t* host_delay,
                        void* dev_workspace, size_t bytes, void* stream);
int spiir_sky_plan_free(spiir_sky_plan* plan);
/* Number of distinct delay tuples of the plan (introspection / DESIGN.md §5). */
int32_t spiir_sky_plan_tuples(const spiir_sky_plan* plan);

/* Result of one (trigger[, slide]) search: the maximum over directions of the
 * coherent SNR^2 (Eq. 9), the pixel where it occurs (on exact ties the first
 * direction in the plan's order: delay tuples in increasing order, pixel index
 * ascending within a tuple), and tot2 = sum_I |z_I|^2, null2 = max(tot2 - coh2, 0) (Eq. 10) there.
 * pix = -1 (and zeros) if the slot is invalid or any gather of the search would
 * leave the valid range of the view. */
typedef struct { float coh2, null2, tot2; int32_t pix; } spiir_sky_result;

/* H5: for every valid trigger (T, t, k) and every direction p:
 *   v_I = z_I[t][k + delay[p][I] - delay[p][T]],
 *   coh2 = sum_j |sum_I U2[p][I][j] v_I|^2 = sum_IJ (U2 U2^T)_IJ Re(v_I conj v_J).
 *   dev_trig [n_slots] (n_slots <= the plan's max_slots); dev_out [n_slots];
 *   dev_skymap (optional, may be NULL) [n_slots][n_pix] coh2 (zeros for slots
 *   with pix = -1). */
int coherent_sky_search(spiir_sky_plan* plan, const spiir_snr_view* view,
                        const spiir_trigger* dev_trig, int32_t n_slots,
                        spiir_sky_result* dev_out, float* dev_skymap, void* stream);

/* H6: the same search for slides s = 1..n_slides with detector I != T read at
 * k - s*step_samples*host_slide_mult[I] + delay difference.
 *   bg_plan may be a coarser table than the foreground's.
 *   dev_out [n_slots][n_slides] (slide s at index s-1). */
int timeslide_background(spiir_sky_plan* bg_plan, const spiir_snr_view* view,
                         const spiir_trigger* dev_trig, int32_t n_slots,
                         int32_t n_slides, int64_t step_samples, const int32_t* host_slide_mult,
                         spiir_sky_result* dev_out, void* stream);
/* NEXT-1 — signal-consistency statistic (Eq. 11 and 12), the second
 * half of the paper's ranking pair (rho_C, xi_C^2).  For every trigger slot with a sky
 * result (pix >= 0):
 *   c_I    = k + delay[pix][I] - delay[pix][T]     (sample of detector I aligned with the trigger)
 *   xi_I^2 = sum_{j=-n_j}^{n_j} |z_I[c_I + j] - z_I[c_I] A[j]|^2 / sum_j (2 - 2 |A[j]|^2)
 *   xi_C^2 = (1/n_det) sum_I xi_I^2
 * with A = dev_autocorr[tmpl][j + n_j], the template's normalised autocorrelation (A[0] = 1).
 * used = 0 and zeros if the slot is invalid, has no pixel, or a window leaves the view.  24 bytes. */
typedef struct { float xi2_c; int32_t used; float xi2[SPIIR_MAX_DET]; } spiir_xi2_result;
/*   dev_delay    [n_pix][n_det] int32, the table handed to spiir_sky_plan_init, on the device
 *   n_slides = 0 : foreground; dev_sky [n_slots] = results of coherent_sky_search for the same dev_trig;
 *                  dev_out [n_slots]
 *   n_slides >= 1: background events; dev_sky [n_slots][n_slides] = results of timeslide_background with the
 *                  same step_samples / host_slide_mult; detector I != T is read n_slides*... earlier exactly as
 *                  there, c_I = k - s*step*mult[I] + delay difference; dev_out [n_slots][n_slides]
 *   dev_autocorr [rows of the view][2 n_j + 1] complex */
int spiir_signal_consistency(const spiir_snr_view* view, int32_t n_det, int32_t n_pix, const int32_t* dev_delay,
                             const spiir_trigger* dev_trig, const spiir_sky_result* dev_sky, int32_t n_slots,
                             int32_t n_slides, int64_t step_samples, const int32_t* host_slide_mult,
                             const spiir_c32* dev_autocorr, int32_t n_j, spiir_xi2_result* dev_out, void* stream);
/* Host helper (float64 inside, set-up only): A[j] = sum_n h[n+j] conj(h[n]) / sum_n |h[n]|^2, j = -n_j..n_j,
 * of the impulse response h[n] = sum_l b_l a_l^(n - d_l) [n >= d_l] of ONE template whose filters all run at
 * the output rate.  host_out [2 n_j + 1]. */
int spiir_template_autocorr(int64_t n_filters, const spiir_c32* host_a, const spiir_c32* host_b,
                            const int32_t* host_delay, int32_t n_j, spiir_c32* host_out);

/* NEXT-2 — ranking statistic and false-alarm probability from the time-slide background
 * (Sec. II D 1).  A background event (trigger, slide) or a foreground candidate is a
 * *coherent event* iff rho_C >= rho_I + sqrt(2) (rho_C = sqrt(coh2), rho_I = trigger snr,
 * decided in float32) and its xi^2 was evaluated (used = 1).  The probability P(rho_C, xi_C^2 | n) of
 * Eq. 13 is a 2-D histogram of the coherent background events; the paper gives no binning: here both axes
 * are uniform in the pseudo-logarithm u(x) = e + (m - 1) of x = m 2^e (m in [1, 2)), x = rho_C^2 on the
 * first axis and xi_C^2 on the second, values outside [u_min, u_max) going to the edge bins.
 *   R(bin)   = (1/N_b) sum of the histogram over bins with rho >= and xi^2 <= this bin's     (Eq. 13)
 *   FAP(bin) = (1/N_b) sum of the histogram over bins whose R is smaller                     (Eq. 14)
 *   FAR      = FAP N_b / T_b                                                                  (Eq. 15)
 * Workspace layout (uint64): [0] N_b, [4 ..) histogram [n_rho][n_xi], then R counts, then FAP counts. */
typedef struct { int32_t n_rho, n_xi; float u_rho_min, u_rho_max, u_xi_min, u_xi_max; } spiir_rank_bins;
typedef struct { float rank, fap, far; int32_t selected; } spiir_rank_result;          /* 16 bytes */
int spiir_rank_workspace_bytes(const spiir_rank_bins* bins, size_t* bytes);
/* Empties the histogram (dev_ws: 16-byte aligned device memory of the queried size). */
int spiir_rank_reset(void* dev_ws, const spiir_rank_bins* bins, void* stream);
/* Adds the coherent events among dev_bg [n_slots][n_slides] (timeslide_background) with their
 * dev_xi [n_slots][n_slides] (spiir_signal_consistency with the same slides) to the histogram. */
int spiir_rank_accumulate(void* dev_ws, const spiir_rank_bins* bins, const spiir_trigger* dev_trig,
                          const spiir_sky_result* dev_bg, const spiir_xi2_result* dev_xi, int32_t n_slots,
                          int32_t n_slides, void* stream);
/* Forms the R and FAP tables from the histogram as it stands (call after accumulating, before ranking). */
int spiir_rank_finalize(void* dev_ws, const spiir_rank_bins* bins, void* stream);
/* Ranks foreground candidates: dev_fg / dev_xi [n_slots] from coherent_sky_search and
 * spiir_signal_consistency; background_seconds = T_b of Eq. 15 (collection time x number of slides);
 * dev_out [n_slots]: zeros and selected = 0 for slots that are not coherent events. */
int spiir_rank_candidates(const void* dev_ws, const spiir_rank_bins* bins, const spiir_trigger* dev_trig,
                          const spiir_sky_result* dev_fg, const spiir_xi2_result* dev_xi, int32_t n_slots,
                          double background_seconds, spiir_rank_result* dev_out, void* stream);

/* The ranking chain of Eq. 13-15 for callers that cannot give it a workspace.
 * Who that is: a search process that reaches the ranking step after all device memory has gone to the filter
 * banks' workspaces and SNR rings (a late cudaMalloc then fails, and where it succeeds it waits for, and holds up,
 * everything in flight on the device — the filtering streams of a low-latency pipeline included), and code that
 * runs inside a host process under a "no device allocation after start-up" rule.
 * One call = spiir_rank_reset + spiir_rank_accumulate(dev_bg_trig, dev_bg, dev_bg_xi, n_bg_slots, n_slides) +
 * spiir_rank_finalize + spiir_rank_candidates(dev_fg_trig, dev_fg, dev_fg_xi, n_fg_slots, background_seconds,
 * dev_out), same kernels, same results bit for bit, with the histogram / R / FAP tables kept in an array that is
 * part of the library image instead of a workspace.  The call itself allocates nothing and frees nothing.
 *   Limit   : n_rho * n_xi <= SPIIR_RANK_STATIC_MAX_BINS, else SPIIR_EINVAL with a message that says so (use the
 *             workspace calls above for finer binnings).  The array is (4 + 3 * 4096) * 8 = 98 336 bytes and every
 *             GPU that loads the library holds it until the process exits.
 *   Set-up  : the first call on each device looks the array's device address up (with that device current, as for
 *             every call); make that first call before any stream capture is begun.
 *   Sharing : one array per device for all callers and streams.  It keeps the last call's tables; the call clears
 *             it before use.  Two calls that overlap on the same GPU (different streams, or different threads) race
 *             on it and give garbage: order them on one stream or with events.
 *   Background from several chunks cannot be accumulated across calls (each call starts from an empty histogram);
 *   pass all events of the collection window in one call.  n_bg_slots = 0 gives an empty background (rank = fap =
 *   far = 0 for every selected candidate); n_fg_slots = 0 only builds the tables.
 *   All dev_* arrays are the caller's, laid out as for the calls above.  Asynchronous on `stream`.
 *   Errors: EINVAL (bins, sizes, NULL pointers, too many bins), ECUDA. */
#define SPIIR_RANK_STATIC_MAX_BINS 4096
int spiir_rank_static(const spiir_rank_bins* bins, const spiir_trigger* dev_bg_trig, const spiir_sky_result* dev_bg,
                      const spiir_xi2_result* dev_bg_xi, int32_t n_bg_slots, int32_t n_slides,
                      const spiir_trigger* dev_fg_trig, const spiir_sky_result* dev_fg,
                      const spiir_xi2_result* dev_fg_xi, int32_t n_fg_slots, double background_seconds,
                      spiir_rank_result* dev_out, void* stream);

/* NEXT-4 — the front end on the device (Sec. II A): FIR down-sampling of the raw
 * strain (16 384 -> 2048 Hz, N_FIR ~ 192 taps), frequency-domain whitening (Eq. 1) against the running median PSD
 * of the immediate past, and amplitude gating with zero padding on either side.  The paper describes the stage in
 * words; the readings W1-W6 are stated in DESIGN.md section 11d:
 *   y[m]   = sum_j taps[j] x[decim m + decim - 1 - j]                                   (x before the stream = 0)
 *   block c = Hann(2 hop) * [hop c-1 | hop c] of y;  D = FFT(block);
 *   S_n[k] = median over the n most recent PAST blocks' periodograms 2 |D[k]|^2 / (f_s sum w^2), n = min(c, n_hist)
 *            made odd, divided by the median bias sum_{i<=n} (-1)^(i+1) / i;  block 0 is not emitted (no past);
 *   d_w    = overlap-add of IFFT(D / sqrt(S_n f_s / 2))                                  (unit variance out)
 *   gate   : |d_w| > gate_threshold zeroes that sample and gate_pad samples on either side.
 * One call consumes ONE hop per detector and returns the `hop` gated samples t in [(c-1) hop - gate_pad,
 * c hop - gate_pad) (zeros before the start of the stream): one hop plus gate_pad of latency.
 * The Fourier transforms are hand-written shared-memory kernels inside the library (no cuFFT). */
typedef struct spiir_frontend spiir_frontend;              /* opaque */
typedef struct {
  int32_t n_det;            /* 1..SPIIR_MAX_DET                                                        */
  int32_t decim;            /* input rate / output rate, 1..16 (paper: 8)                              */
  int32_t n_taps;           /* 1..512 and <= hop * decim (paper: ~192)                                 */
  int32_t hop;              /* output samples per call, a power of two in 256..4096 (paper: 2 s = 4096) */
  int32_t n_hist;           /* PSD history in blocks, 1..31 (paper: 56 s of 4-s blocks at a 2-s hop = 27) */
  int32_t gate_pad;         /* output samples zeroed on either side of an excursion, <= hop / 2 (paper: 0.25 s = 512) */
  float   out_rate_hz;      /* f_s of the output (2048)                                               */
  float   gate_threshold;   /* in units of the whitened standard deviation                            */
  const float* host_taps;   /* [n_taps], copied at init                                               */
} spiir_frontend_desc;
int spiir_frontend_workspace_bytes(const spiir_frontend_desc* desc, size_t* bytes);
/* dev_workspace: 256-byte aligned, alive until spiir_frontend_free.  Synchronises the stream once (set-up). */
int spiir_frontend_init(spiir_frontend** out, const spiir_frontend_desc* desc, void* dev_workspace, size_t bytes, void* stream);
int spiir_frontend_reset(spiir_frontend* fe, void* stream);        /* back to the start of a stream */
int spiir_frontend_free(spiir_frontend* fe);
/*   dev_raw [n_det][hop * decim] float32; dev_out [n_det][hop] float32; dev_psd (optional, may be NULL)
 *   [n_det][hop + 1]: the S_n used for this block (zeros for block 0).  Asynchronous on `stream`. */
int spiir_frontend_chunk(spiir_frontend* fe, const float* dev_raw, float* dev_out, float* dev_psd, void* stream);

/* Introspection: the layout chosen for a band (lanes per unit G, filters per lane
 * F, units, padded slots, shared-memory history depth) and counters for bench. */
typedef struct {
  int32_t lanes_per_unit, filters_per_lane, n_units, n_units_long;
  int32_t smem_history, smem_bytes;
  int64_t n_filters, n_slots;
} spiir_band_plan;
int spiir_bank_band_plan(const spiir_bank* bank, int32_t band, spiir_band_plan* plan);
/* Filter-sample updates (real filters only, all detectors) one chunk of n_samples performs. */
int64_t spiir_bank_updates_per_chunk(const spiir_bank* bank, int32_t n_samples);
/* Kernels launched by this library on this thread so far (bench bookkeeping). */
int64_t spiir_launch_count(void);

/* Profiling aid for bench.py (off by default; the hot path records no events when
 * off).  spiir_bank_timing_enable(bank, n_chunks) with n_chunks >= 1 creates the
 * CUDA events for n_chunks calls (the only place events are created — never inside
 * spiir_filter_chunk) and switches recording on: each of the next n_chunks
 * spiir_filter_chunk calls records events on the caller's stream at its begin and
 * end and around its recursion-kernel launches (k_bank); further calls go
 * unrecorded.  n_chunks = 0 switches it off.
 * spiir_bank_timing_read synchronises those events, returns the summed durations
 * (ms) of the recursion brackets and of the whole calls and the number of calls
 * recorded since the last read, and clears the record (the enabled count stands). */
int spiir_bank_timing_enable(spiir_bank* bank, int32_t n_chunks);
int spiir_bank_timing_read(spiir_bank* bank, double* ms_recursion, double* ms_chunk, int32_t* n_chunks);

const char* spiir_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SPIIR_H */
