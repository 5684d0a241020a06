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
#include "spiir_internal.cuh"

namespace spiir {

constexpr int kUpThreads = 128;
constexpr int kUpMaxFactor = 16;

struct UpParams {
  const float2* z; int64_t det_stride, row_stride, ring_len, k_newest, n_rows;
  const spiir_trigger* trig; int32_t n_slots, n_det;
  int32_t R, H, Lw; int64_t Lp;
  float4 w[kUpMaxFactor];
  float2* out; spiir_trigger* trig_out;
};

// the re-addressed candidates (one thread per slot)
__global__ void __launch_bounds__(kUpThreads) k_upsample_trig(const __grid_constant__ UpParams P) {
  const int s = blockIdx.x * kUpThreads + threadIdx.x;
  if (s >= P.n_slots) return;
  const spiir_trigger t = P.trig[s];
  const int64_t k_old = P.k_newest - P.ring_len + 1 > 0 ? P.k_newest - P.ring_len + 1 : 0;
  const bool ok = t.valid && t.tmpl >= 0 && t.tmpl < P.n_rows && t.k - P.H - 1 >= k_old && t.k + P.H + 1 <= P.k_newest;
  spiir_trigger o = t;
  o.valid = ok ? 1 : 0; o.tmpl = s; o.k = (int64_t)P.R * P.H;
  if (!t.valid) { o.det = 0; o.z_re = o.z_im = o.snr = 0.f; }
  o._pad = 0; o._pad2 = 0.f;
  P.trig_out[s] = o;
}

// the windows: one CTA per (slot, detector), threads stride over the output samples (coalesced stores; the
// 2 H + 3 ring samples a window reads are consecutive and stay in L1 across the R phases).  One 64-bit
// modulo per thread places the window in the ring; after that a sample's neighbours are conditional wraps.
__global__ void __launch_bounds__(kUpThreads) k_upsample(const __grid_constant__ UpParams P) {
  const int s = blockIdx.x, I = blockIdx.y;
  const spiir_trigger t = P.trig[s];
  const int64_t k_old = P.k_newest - P.ring_len + 1 > 0 ? P.k_newest - P.ring_len + 1 : 0;
  const bool ok = t.valid && t.tmpl >= 0 && t.tmpl < P.n_rows && t.k - P.H - 1 >= k_old && t.k + P.H + 1 <= P.k_newest;
  float2* out = P.out + ((size_t)I * P.n_slots + s) * P.Lp;
  if (!ok) {
    for (int u = threadIdx.x; u < P.Lp; u += kUpThreads) out[u] = make_float2(0.f, 0.f);
    return;
  }
  const float2* zr = P.z + (size_t)I * P.det_stride + (size_t)t.tmpl * P.row_stride;
  const int64_t L = P.ring_len;
  const int64_t i0 = (t.k - P.H) % L;                    // t.k - H >= 1 here
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

int spiir_snr_upsample_windows(const spiir_snr_view* view, int32_t n_det, const spiir_trigger* dev_trig,
                               int32_t n_slots, int32_t factor, int32_t half_width, spiir_c32* dev_out,
                               spiir_trigger* dev_trig_out, spiir_snr_view* out_view, void* stream) {
  size_t elems = 0;
  int rc = spiir_snr_upsample_elems(n_det, n_slots, factor, half_width, &elems);
  if (rc) return rc;
  SPIIR_REQUIRE(view && view->dev_z && dev_trig && dev_out && dev_trig_out && out_view, "a pointer is NULL");
  SPIIR_REQUIRE(view->ring_len >= 1 && view->k_newest >= 0 && view->n_rows >= 1, "bad view");
  SPIIR_REQUIRE(((uintptr_t)dev_out & 15) == 0, "dev_out must be 16-byte aligned");
  UpParams P;
  P.z = (const float2*)view->dev_z;
  P.det_stride = view->det_stride; P.row_stride = view->row_stride;
  P.ring_len = view->ring_len; P.k_newest = view->k_newest; P.n_rows = view->n_rows;
  P.trig = dev_trig; P.n_slots = n_slots; P.n_det = n_det;
  P.R = factor; P.H = half_width; P.Lw = 2 * factor * half_width + 1;
  P.Lp = ((int64_t)P.Lw + 1) & ~(int64_t)1;
  for (int r = 0; r < kUpMaxFactor; ++r) {
    // cubic through nodes -1, 0, 1, 2 evaluated at mu = r / R, in float64, rounded once
    const double m = r < factor ? (double)r / factor : 0.0;
    P.w[r] = make_float4((float)(-m * (m - 1.0) * (m - 2.0) / 6.0), (float)((m + 1.0) * (m - 1.0) * (m - 2.0) / 2.0),
                         (float)(-(m + 1.0) * m * (m - 2.0) / 2.0), (float)((m + 1.0) * m * (m - 1.0) / 6.0));
  }
  P.out = (float2*)dev_out; P.trig_out = dev_trig_out;
  out_view->dev_z = dev_out;
  out_view->det_stride = (int64_t)n_slots * P.Lp;
  out_view->row_stride = P.Lp;
  out_view->ring_len = P.Lp;
  out_view->k_newest = P.Lw - 1;
  out_view->n_rows = n_slots;
  if (n_slots == 0) return SPIIR_OK;
  k_upsample_trig<<<(n_slots + kUpThreads - 1) / kUpThreads, kUpThreads, 0, (cudaStream_t)stream>>>(P);
  k_upsample<<<dim3((unsigned)n_slots, (unsigned)n_det), kUpThreads, 0, (cudaStream_t)stream>>>(P);
  count_launch(2);
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

}  // extern "C"
