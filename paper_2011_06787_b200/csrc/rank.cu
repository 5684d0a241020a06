// NEXT-2 — ranking statistic and false-alarm probability from the time-slide background
// (Sec. II D 1):
//   selection   rho_C >= rho_I + sqrt(2)
//   P(rho_C, xi_C^2 | n)   2-D histogram of the selected background events
//   R(rho', xi') = sum_{rho >= rho', xi^2 <= xi'} P                           (Eq. 13, at bin granularity)
//   FAP(R') = sum_{R < R'} P(R | n)                                           (Eq. 14)
//   FAR = FAP N_b / T_b                                                       (Eq. 15)
// The paper gives no binning; reading X3: uniform bins in the pseudo-logarithm
// u(x) = e + (m - 1), x = m 2^e, read off the float32 bit pattern, so that a bin is decided by a
// handful of float32 operations and no transcendental function.  All sums are integer counts
// (64-bit); R and FAP are ordered and compared as counts, and reported as count / N_b.
//
//   k_rank_hist    thread = background event: cut, bin, atomicAdd          (HBM-bound, 36 B per event)
//   k_rank_rows    C1[i][j] = sum_{j' <= j} H[i][j']     (thread = row)
//   k_rank_cols    C[i][j]  = sum_{i' >= i} C1[i'][j]    (thread = column)
//   k_rank_fap     F[b] = sum_{b': C[b'] < C[b]} H[b']   (thread = bin, all bins streamed through
//                  shared memory: n_bins^2 compare-adds, the plain definition)
//   k_rank_lookup  thread = foreground candidate
#include "spiir_internal.cuh"

#include <mutex>

namespace spiir {

typedef unsigned long long u64;

struct RankWs { u64* H; u64* C; u64* F; u64* nb; };

static size_t rank_bins_total(const spiir_rank_bins* b) { return (size_t)b->n_rho * b->n_xi; }
static RankWs rank_carve(void* ws, const spiir_rank_bins* b) {
  const size_t n = rank_bins_total(b);
  RankWs r;
  r.nb = (u64*)ws;                       // [0] = N_b (32 bytes reserved)
  r.H = r.nb + 4; r.C = r.H + n; r.F = r.C + n;
  return r;
}

struct RankAxis { float u_min, scale; int n; };

__device__ __forceinline__ int rank_bin(float x, RankAxis a) {
  if (!(x > 0.f)) return 0;
  const float u = __int2float_rn(__float_as_int(x) - 0x3F800000) * 1.1920928955078125e-07f;   // 2^-23
  const float t = floorf(__fmul_rn(__fsub_rn(u, a.u_min), a.scale));
  return (int)fminf(fmaxf(t, 0.f), (float)(a.n - 1));
}
__device__ __forceinline__ bool rank_selected(float snr_trig, float coh2, int used) {
  return used != 0 && __fsqrt_rn(coh2) >= __fadd_rn(snr_trig, 1.41421356f);
}

__global__ void __launch_bounds__(256) k_rank_hist(const spiir_trigger* trig, const spiir_sky_result* bg,
                                                   const spiir_xi2_result* xi, long long n_events, int S1,
                                                   RankAxis ar, RankAxis ax, u64* H, u64* nb) {
  const long long e = (long long)blockIdx.x * 256 + threadIdx.x;
  bool sel = false;
  if (e < n_events) {
    const spiir_xi2_result x = xi[e];
    const spiir_sky_result r = bg[e];
    const float snr = trig[e / S1].snr;
    sel = r.pix >= 0 && rank_selected(snr, r.coh2, x.used);
    if (sel) atomicAdd(H + (size_t)rank_bin(r.coh2, ar) * ax.n + rank_bin(x.xi2_c, ax), 1ull);
  }
  const unsigned m = __ballot_sync(0xffffffffu, sel);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(nb, (u64)__popc(m));
}

__global__ void k_rank_rows(const u64* H, u64* C, int n_rho, int n_xi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_rho) return;
  u64 s = 0;
  for (int j = 0; j < n_xi; ++j) { s += H[(size_t)i * n_xi + j]; C[(size_t)i * n_xi + j] = s; }
}
__global__ void k_rank_cols(u64* C, int n_rho, int n_xi) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_xi) return;
  u64 s = 0;
  for (int i = n_rho - 1; i >= 0; --i) { s += C[(size_t)i * n_xi + j]; C[(size_t)i * n_xi + j] = s; }
}

constexpr int kFapThreads = 256;
__global__ void __launch_bounds__(kFapThreads) k_rank_fap(const u64* H, const u64* C, u64* F, int n) {
  __shared__ u64 sc[kFapThreads], sh[kFapThreads];
  const int b = blockIdx.x * kFapThreads + threadIdx.x;
  const u64 mine = b < n ? C[b] : 0ull;
  u64 acc = 0;
  for (int t0 = 0; t0 < n; t0 += kFapThreads) {
    const int q = t0 + threadIdx.x;
    __syncthreads();
    sc[threadIdx.x] = q < n ? C[q] : ~0ull;          // padding never counts: nothing is < it ... and H = 0
    sh[threadIdx.x] = q < n ? H[q] : 0ull;
    __syncthreads();
#pragma unroll 8
    for (int k = 0; k < kFapThreads; ++k) acc += sc[k] < mine ? sh[k] : 0ull;
  }
  if (b < n) F[b] = acc;
}

__global__ void __launch_bounds__(256) k_rank_lookup(const spiir_trigger* trig, const spiir_sky_result* fg,
                                                     const spiir_xi2_result* xi, int n_slots, RankAxis ar,
                                                     RankAxis ax, const u64* C, const u64* F, const u64* nb,
                                                     double t_b, spiir_rank_result* out) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= n_slots) return;
  spiir_rank_result res; res.rank = 0.f; res.fap = 0.f; res.far = 0.f; res.selected = 0;
  const spiir_trigger t = trig[i];
  const spiir_sky_result r = fg[i];
  const spiir_xi2_result x = xi[i];
  if (t.valid && r.pix >= 0 && rank_selected(t.snr, r.coh2, x.used)) {
    const size_t b = (size_t)rank_bin(r.coh2, ar) * ax.n + rank_bin(x.xi2_c, ax);
    const double n_b = (double)nb[0];
    res.selected = 1;
    if (n_b > 0) {
      res.rank = (float)((double)C[b] / n_b);
      res.fap = (float)((double)F[b] / n_b);
      res.far = (float)((double)F[b] / t_b);           // FAP * N_b / T_b
    }
  }
  out[i] = res;
}

static int rank_check(const spiir_rank_bins* b) {
  SPIIR_REQUIRE(b != nullptr, "bins is NULL");
  SPIIR_REQUIRE(b->n_rho >= 1 && b->n_xi >= 1 && (long long)b->n_rho * b->n_xi <= (1 << 22), "bad bin counts");
  SPIIR_REQUIRE(b->u_rho_max > b->u_rho_min && b->u_xi_max > b->u_xi_min, "empty bin range");
  return SPIIR_OK;
}
static RankAxis axis(float lo, float hi, int n) {
  RankAxis a; a.u_min = lo; a.n = n;
  a.scale = (float)n / (hi - lo);                      // float32 division, as the oracle's
  return a;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

int spiir_rank_workspace_bytes(const spiir_rank_bins* bins, size_t* bytes) {
  int rc = rank_check(bins);
  if (rc) return rc;
  SPIIR_REQUIRE(bytes != nullptr, "bytes is NULL");
  *bytes = (4 + 3 * rank_bins_total(bins)) * sizeof(u64);
  return SPIIR_OK;
}

int spiir_rank_reset(void* dev_ws, const spiir_rank_bins* bins, void* stream) {
  int rc = rank_check(bins);
  if (rc) return rc;
  SPIIR_REQUIRE(dev_ws != nullptr && ((uintptr_t)dev_ws & 15) == 0, "workspace NULL or misaligned");
  SPIIR_CUDA_OK(cudaMemsetAsync(dev_ws, 0, (4 + 3 * rank_bins_total(bins)) * sizeof(u64), (cudaStream_t)stream));
  return SPIIR_OK;
}

int spiir_rank_accumulate(void* dev_ws, const spiir_rank_bins* bins, const spiir_trigger* dev_trig,
                          const spiir_sky_result* dev_bg, const spiir_xi2_result* dev_xi, int32_t n_slots,
                          int32_t n_slides, void* stream) {
  int rc = rank_check(bins);
  if (rc) return rc;
  SPIIR_REQUIRE(dev_ws && dev_trig && dev_bg && dev_xi, "a pointer is NULL");
  SPIIR_REQUIRE(n_slots >= 0 && n_slides >= 1, "bad n_slots / n_slides");
  const long long n_ev = (long long)n_slots * n_slides;
  if (n_ev == 0) return SPIIR_OK;
  const RankWs w = rank_carve(dev_ws, bins);
  k_rank_hist<<<(unsigned)((n_ev + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      dev_trig, dev_bg, dev_xi, n_ev, n_slides, axis(bins->u_rho_min, bins->u_rho_max, bins->n_rho),
      axis(bins->u_xi_min, bins->u_xi_max, bins->n_xi), w.H, w.nb);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

int spiir_rank_finalize(void* dev_ws, const spiir_rank_bins* bins, void* stream) {
  int rc = rank_check(bins);
  if (rc) return rc;
  SPIIR_REQUIRE(dev_ws != nullptr, "workspace is NULL");
  const RankWs w = rank_carve(dev_ws, bins);
  const int n = (int)rank_bins_total(bins);
  cudaStream_t st = (cudaStream_t)stream;
  k_rank_rows<<<(bins->n_rho + 127) / 128, 128, 0, st>>>(w.H, w.C, bins->n_rho, bins->n_xi);
  k_rank_cols<<<(bins->n_xi + 127) / 128, 128, 0, st>>>(w.C, bins->n_rho, bins->n_xi);
  k_rank_fap<<<(n + kFapThreads - 1) / kFapThreads, kFapThreads, 0, st>>>(w.H, w.C, w.F, n);
  count_launch(3);
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

int spiir_rank_candidates(const void* dev_ws, const spiir_rank_bins* bins, const spiir_trigger* dev_trig,
                          const spiir_sky_result* dev_fg, const spiir_xi2_result* dev_xi, int32_t n_slots,
                          double background_seconds, spiir_rank_result* dev_out, void* stream) {
  int rc = rank_check(bins);
  if (rc) return rc;
  SPIIR_REQUIRE(dev_ws && dev_trig && dev_fg && dev_xi && dev_out, "a pointer is NULL");
  SPIIR_REQUIRE(n_slots >= 0 && background_seconds > 0, "bad n_slots / background_seconds");
  if (n_slots == 0) return SPIIR_OK;
  const RankWs w = rank_carve(const_cast<void*>(dev_ws), bins);
  k_rank_lookup<<<(n_slots + 255) / 256, 256, 0, (cudaStream_t)stream>>>(
      dev_trig, dev_fg, dev_xi, n_slots, axis(bins->u_rho_min, bins->u_rho_max, bins->n_rho),
      axis(bins->u_xi_min, bins->u_xi_max, bins->n_xi), w.C, w.F, w.nb, background_seconds, dev_out);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------
// spiir_rank_static — the whole ranking chain in one call that needs no workspace from the caller.
//
// Every other spiir_rank_* call works on a workspace the caller has to allocate (histogram, R counts, FAP
// counts).  An online search process cannot always do that when the ranking step is reached: by then it has
// usually handed all of the GPU's memory to the filter banks' workspaces and SNR rings, so a late cudaMalloc
// fails; and where it would succeed it serialises against all work in flight on the device and holds up the
// filtering streams, which a low-latency pipeline cannot afford.  Plug-ins that run inside somebody else's
// process under a "no device allocation after start-up" rule are in the same position.
//
// The tables therefore live in the array below, which is part of the library image: every GPU that loads
// libspiir_b200.so carries these (4 + 3 * SPIIR_RANK_STATIC_MAX_BINS) * 8 = 98 336 bytes until the process exits.
// There is ONE array per device, shared by every call whatever its stream, and it keeps what the last call left
// in it; the call clears it first, and two calls that overlap on the same GPU race on it.
//
// g_rank_static is a device symbol.  In host code the name is only a handle: taking its address there does not
// yield device memory (a kernel handed that value faults, or reads host memory where the GPU can reach it).  The
// device address is asked for once per device with cudaGetSymbolAddress and kept in rank_static_ptr().
namespace spiir {

constexpr size_t kRankStaticWords = 4 + 3 * (size_t)SPIIR_RANK_STATIC_MAX_BINS;
static __device__ __align__(256) u64 g_rank_static[kRankStaticWords];

constexpr int kRankStaticMaxDevices = 64;

// Device address of g_rank_static on the CURRENT device.  The first call on a device resolves the symbol (which
// may make the runtime load the module there); later calls only read the cached pointer.
static int rank_static_ptr(u64** out) {
  static std::mutex mu;
  static u64* ptr[kRankStaticMaxDevices] = {};
  int dev = -1;
  SPIIR_CUDA_OK(cudaGetDevice(&dev));
  SPIIR_REQUIRE(dev >= 0 && dev < kRankStaticMaxDevices, "spiir_rank_static: device ordinal %d is outside 0..%d", dev,
                kRankStaticMaxDevices - 1);
  std::lock_guard<std::mutex> lock(mu);
  if (ptr[dev] == nullptr) {
    void* p = nullptr;
    SPIIR_CUDA_OK(cudaGetSymbolAddress(&p, g_rank_static));
    if (p == nullptr) {
      set_error("spiir_rank_static: cudaGetSymbolAddress returned a null address on device %d", dev);
      return SPIIR_ECUDA;
    }
    ptr[dev] = (u64*)p;
  }
  *out = ptr[dev];
  return SPIIR_OK;
}

}  // namespace spiir

extern "C" {

int spiir_rank_static(const spiir_rank_bins* bins, const spiir_trigger* dev_bg_trig, const spiir_sky_result* dev_bg,
                      const spiir_xi2_result* dev_bg_xi, int32_t n_bg_slots, int32_t n_slides,
                      const spiir_trigger* dev_fg_trig, const spiir_sky_result* dev_fg,
                      const spiir_xi2_result* dev_fg_xi, int32_t n_fg_slots, double background_seconds,
                      spiir_rank_result* dev_out, void* stream) {
  int rc = rank_check(bins);
  if (rc) return rc;
  const size_t n = rank_bins_total(bins);
  SPIIR_REQUIRE(n <= (size_t)SPIIR_RANK_STATIC_MAX_BINS,
                "spiir_rank_static: n_rho * n_xi = %zu bins exceed the built-in table of SPIIR_RANK_STATIC_MAX_BINS = %d; "
                "use spiir_rank_accumulate / _finalize / _candidates with a workspace of your own",
                n, SPIIR_RANK_STATIC_MAX_BINS);
  SPIIR_REQUIRE(n_bg_slots >= 0 && n_slides >= 1 && n_fg_slots >= 0 && background_seconds > 0,
                "bad n_bg_slots / n_slides / n_fg_slots / background_seconds");
  const long long n_ev = (long long)n_bg_slots * n_slides;
  SPIIR_REQUIRE(n_ev == 0 || (dev_bg_trig && dev_bg && dev_bg_xi), "a background pointer is NULL");
  SPIIR_REQUIRE(n_fg_slots == 0 || (dev_fg_trig && dev_fg && dev_fg_xi && dev_out), "a foreground pointer is NULL");
  u64* scratch = nullptr;
  rc = rank_static_ptr(&scratch);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const RankWs w = rank_carve(scratch, bins);
  const RankAxis ar = axis(bins->u_rho_min, bins->u_rho_max, bins->n_rho);
  const RankAxis ax = axis(bins->u_xi_min, bins->u_xi_max, bins->n_xi);
  // the array still holds the previous call's tables: N_b and the histogram are summed into, so they start at zero
  // (R and FAP counts are overwritten in full by k_rank_rows / k_rank_fap, cleared all the same)
  SPIIR_CUDA_OK(cudaMemsetAsync(scratch, 0, (4 + 3 * n) * sizeof(u64), st));
  if (n_ev > 0) {
    k_rank_hist<<<(unsigned)((n_ev + 255) / 256), 256, 0, st>>>(dev_bg_trig, dev_bg, dev_bg_xi, n_ev, n_slides, ar, ax,
                                                                w.H, w.nb);
    count_launch();
  }
  k_rank_rows<<<(bins->n_rho + 127) / 128, 128, 0, st>>>(w.H, w.C, bins->n_rho, bins->n_xi);
  k_rank_cols<<<(bins->n_xi + 127) / 128, 128, 0, st>>>(w.C, bins->n_rho, bins->n_xi);
  k_rank_fap<<<((int)n + kFapThreads - 1) / kFapThreads, kFapThreads, 0, st>>>(w.H, w.C, w.F, (int)n);
  count_launch(3);
  if (n_fg_slots > 0) {
    k_rank_lookup<<<(n_fg_slots + 255) / 256, 256, 0, st>>>(dev_fg_trig, dev_fg, dev_fg_xi, n_fg_slots, ar, ax, w.C,
                                                            w.F, w.nb, background_seconds, dev_out);
    count_launch();
  }
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

}  // extern "C"
