// NEXT-1 — signal-consistency statistic xi^2 (Eq. 11 and 12):
//   xi_I^2 = sum_{j=-nj}^{nj} |z_I[c_I + j] - z_I[c_I] A[j]|^2 / sum_j (2 - 2 |A[j]|^2),
//   xi_C^2 = (1/N_d) sum_I xi_I^2,
// A = the template's normalised autocorrelation, c_I = the sample of detector I aligned with
// the trigger at the direction the coherent search returned (reading X1).
// One warp per trigger slot: lanes stride over the 2 nj + 1 lags (coalesced reads of the SNR
// ring and of the autocorrelation row), warp-shuffle sums.  HBM-bound: ~(N_d + 1) x 2.8 KB per
// candidate at nj = 175.
#include <cmath>
#include <complex>
#include <vector>

#include "spiir_internal.cuh"

namespace spiir {

constexpr int kXiThreads = 128;

struct Xi2Params {
  const float2* z; int64_t det_stride, row_stride, ring_len, k_newest, n_rows;
  const spiir_trigger* trig; const spiir_sky_result* sky; int32_t n_slots;
  const int32_t* delay; int32_t n_det, n_pix;
  const float2* acorr; int32_t nj;
  int32_t n_slides; int64_t step; int32_t mult[SPIIR_MAX_DET];   // n_slides = 0: foreground
  spiir_xi2_result* out;
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void __launch_bounds__(kXiThreads) k_xi2(const __grid_constant__ Xi2Params P) {
  const int lane = threadIdx.x & 31;
  const int S1 = P.n_slides > 0 ? P.n_slides : 1;
  const long long w = (long long)blockIdx.x * (kXiThreads / 32) + (threadIdx.x >> 5);   // (slot, slide)
  if (w >= (long long)P.n_slots * S1) return;
  const int i = (int)(w / S1), sl = (int)(w - (long long)i * S1) + (P.n_slides > 0 ? 1 : 0);
  spiir_xi2_result res;
  res.xi2_c = 0.f; res.used = 0;
#pragma unroll
  for (int I = 0; I < SPIIR_MAX_DET; ++I) res.xi2[I] = 0.f;
  const spiir_trigger tr = P.trig[i];
  const int pix = P.sky[w].pix;
  const int D = P.n_det, nj = P.nj, W = 2 * nj + 1;
  bool ok = tr.valid && pix >= 0 && pix < P.n_pix && tr.det >= 0 && tr.det < D && tr.tmpl >= 0 && tr.tmpl < P.n_rows;
  int64_t c[SPIIR_MAX_DET];
  if (ok) {
    const int64_t kmin = (P.k_newest - P.ring_len + 1 > 0) ? P.k_newest - P.ring_len + 1 : 0;
    const int32_t* dl = P.delay + (size_t)pix * D;
    const int dT = __ldg(dl + tr.det);
    for (int I = 0; I < D; ++I) {
      c[I] = tr.k + (int64_t)__ldg(dl + I) - dT - (I != tr.det ? (int64_t)sl * P.step * P.mult[I] : 0);
      ok = ok && c[I] - nj >= kmin && c[I] + nj <= P.k_newest;
    }
  }
  if (ok) {
    const float2* A = P.acorr + (size_t)tr.tmpl * W;
    float den = 0.f;
    for (int j = lane; j < W; j += 32) {
      const float2 a = __ldg(A + j);
      den += 2.f - 2.f * fmaf(a.x, a.x, a.y * a.y);
    }
    den = warp_sum(den);
    float mean = 0.f;
    for (int I = 0; I < D; ++I) {
      const float2* zr = P.z + (size_t)I * P.det_stride + (size_t)tr.tmpl * P.row_stride;
      const float2 z0 = zr[c[I] % P.ring_len];
      int64_t idx = (c[I] - nj + lane) % P.ring_len;
      float num = 0.f;
      for (int j = lane; j < W; j += 32) {
        const float2 a = __ldg(A + j);
        const float2 v = zr[idx];
        const float er = v.x - (z0.x * a.x - z0.y * a.y), ei = v.y - (z0.x * a.y + z0.y * a.x);
        num = fmaf(er, er, fmaf(ei, ei, num));
        idx += 32;
        if (idx >= P.ring_len) idx -= P.ring_len;
      }
      num = warp_sum(num);
      const float x = den > 0.f ? num / den : 0.f;
      res.xi2[I] = x;
      mean += x;
    }
    res.xi2_c = mean / (float)D;
    res.used = 1;
  }
  if (lane == 0) P.out[w] = res;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

int spiir_signal_consistency(const spiir_snr_view* view, int32_t n_det, int32_t n_pix, const int32_t* dev_delay,
                             const spiir_trigger* dev_trig, const spiir_sky_result* dev_sky, int32_t n_slots,
                             int32_t n_slides, int64_t step_samples, const int32_t* host_slide_mult,
                             const spiir_c32* dev_autocorr, int32_t n_j, spiir_xi2_result* dev_out, void* stream) {
  SPIIR_REQUIRE(dev_delay && dev_trig && dev_sky && dev_autocorr && dev_out, "a pointer is NULL");
  if (int rcv = check_snr_view(view)) return rcv;
  SPIIR_REQUIRE(n_det >= 1 && n_det <= SPIIR_MAX_DET, "n_det %d out of range", n_det);
  SPIIR_REQUIRE(n_pix >= 1 && n_slots >= 0 && n_j >= 1, "bad n_pix / n_slots / n_j");
  SPIIR_REQUIRE(2 * (int64_t)n_j + 1 <= view->ring_len, "window of %d lags longer than the view", 2 * n_j + 1);
  if (int rcs = check_slides(n_slides, step_samples, host_slide_mult, n_det)) return rcs;
  if (n_slots == 0) return SPIIR_OK;
  Xi2Params P;
  P.z = (const float2*)view->dev_z; P.det_stride = view->det_stride; P.row_stride = view->row_stride;
  P.ring_len = view->ring_len; P.k_newest = view->k_newest; P.n_rows = view->n_rows;
  P.trig = dev_trig; P.sky = dev_sky; P.n_slots = n_slots;
  P.delay = dev_delay; P.n_det = n_det; P.n_pix = n_pix;
  P.acorr = (const float2*)dev_autocorr; P.nj = n_j; P.out = dev_out;
  P.n_slides = n_slides; P.step = step_samples;
  for (int I = 0; I < SPIIR_MAX_DET; ++I) P.mult[I] = (n_slides > 0 && I < n_det) ? host_slide_mult[I] : 0;
  const int wpb = kXiThreads / 32;
  const long long n_w = (long long)n_slots * (n_slides > 0 ? n_slides : 1);
  k_xi2<<<(unsigned)((n_w + wpb - 1) / wpb), kXiThreads, 0, (cudaStream_t)stream>>>(P);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

// Host helper (float64, set-up only): impulse response of one single-band template by the recursion
// itself, then the lag sums written out.
int spiir_template_autocorr(int64_t n_filters, const spiir_c32* host_a, const spiir_c32* host_b,
                            const int32_t* host_delay, int32_t n_j, spiir_c32* host_out) {
  SPIIR_REQUIRE(n_filters >= 1 && host_a && host_b && host_delay && host_out && n_j >= 1, "bad arguments");
  typedef std::complex<double> cd;
  int dmax = 0; double tau_max = 1.0;
  for (int64_t l = 0; l < n_filters; ++l) {
    const cd a(host_a[l].re, host_a[l].im);
    SPIIR_REQUIRE(std::abs(a) < 1.0 && std::abs(a) > 0.0, "filter %lld: |a| must be in (0, 1)", (long long)l);
    SPIIR_REQUIRE(host_delay[l] >= 0, "filter %lld: negative delay", (long long)l);
    dmax = std::max(dmax, (int)host_delay[l]);
    tau_max = std::max(tau_max, -1.0 / std::log(std::abs(a)));
  }
  const int64_t N = dmax + (int64_t)std::ceil(25.0 * tau_max) + n_j + 8;
  std::vector<cd> h((size_t)N, cd(0, 0));
  for (int64_t l = 0; l < n_filters; ++l) {
    const cd a(host_a[l].re, host_a[l].im), b(host_b[l].re, host_b[l].im);
    cd y = b;                                            // y[d] = b, y[n] = a y[n-1]
    for (int64_t n = host_delay[l]; n < N; ++n) { h[(size_t)n] += y; y *= a; }
  }
  double norm = 0;
  for (int64_t n = 0; n < N; ++n) norm += std::norm(h[(size_t)n]);
  SPIIR_REQUIRE(norm > 0, "template has zero response");
  for (int j = -n_j; j <= n_j; ++j) {
    cd r(0, 0);
    const int64_t n0 = j >= 0 ? 0 : -j;                  // sum_n h[n + j] conj(h[n])
    for (int64_t n = n0; n + j < N && n < N; ++n) r += h[(size_t)(n + j)] * std::conj(h[(size_t)n]);
    r /= norm;
    host_out[j + n_j].re = (float)r.real(); host_out[j + n_j].im = (float)r.imag();
  }
  return SPIIR_OK;
}

}  // extern "C"
