// H5 / H6 — coherent sky-direction search and its time-slide background for sm_100a.
//
// PAPER.md:147-157 (Eq. 9, 10): rho_c^2 = || I U^T z ||^2, rho_null^2 = sum |z_I|^2 - rho_c^2,
// evaluated for every candidate on every HEALPix direction with the
// per-direction look-up tables of U and the time offsets; background
// from time-shifted companions.
//
// Design — not the paper's "one thread per direction":
//   * Eq. 28 writes rho_c^2 as the quadratic form z^H (U I U^T) z.  With
//     integer delays only ~N_pix/14 distinct delay tuples exist at nside 64, and every
//     direction of one tuple gathers the SAME samples.  So the plan sorts directions
//     by tuple and stores the projector M = U2 U2^T; per tuple a thread forms the
//     N_d(N_d+1)/2 real products q_IJ = Re(z_I conj z_J) once, and each direction then
//     costs one N_q-term dot product (6 FP32 instructions for three detectors)
//     plus the running arg-max.
//   * thread = K (trigger, slide) pairs; a CTA owns 32 K pairs whose delay windows
//     (the only samples any direction can touch) sit in shared memory, sample-major
//     so that the per-tuple gather is conflict free; its warps split the direction
//     stream and stage their records through shared memory for broadcast reads.
//   * valid trigger slots are binned by trigger detector on the device (no host sync);
//     one launch per trigger detector, persistent CTAs stride over the pair batches.
#include <algorithm>
#include <climits>
#include <cstring>
#include <vector>

#include "spiir_internal.cuh"

namespace spiir {

constexpr int kSkyThreads = 256;
constexpr int kSkyWarps = kSkyThreads / 32;
constexpr int kSkyK = 2;                    // pairs per thread
constexpr int kSkyNP = 32 * kSkyK;          // pairs per CTA
constexpr int kSkyNPS = kSkyNP + 1;         // padded row stride of the windows (float2)
constexpr int kSkySmemMax = 200 * 1024;

template <int D> struct SkyRec { static constexpr int NQ = D * (D + 1) / 2; static constexpr int RW = (NQ + 3 + 3) / 4 * 4; };
// record words: [0, NQ) projector entries (diagonal first, then 2*M_IJ for I<J in the
// order (0,1) (0,2) (1,2) (0,3) (1,3) (2,3)); [NQ] pixel; [NQ+1] d1 | d2 << 16; [NQ+2] d3
// with d_I = delay[p][I] - delay[p][0].

struct SkyParams {
  const float* rec; int32_t n_rec; int32_t rec_per_warp;     // stream, multiple-of-32 share per warp
  const int32_t* pix_delta;                                   // [n_pix][4] d_I of each pixel (word 0 unused)
  int32_t n_pix;
  const float2* z; int64_t det_stride, row_stride, ring_len, k_newest;
  const spiir_trigger* trig;
  const int32_t* list; const int32_t* counts;                 // this launch: list of slots of trigger detector T
  int32_t T;                                                  // trigger detector
  int32_t n_slides;                                           // 0 = foreground
  int64_t step; int32_t mult[SPIIR_MAX_DET];
  int32_t lo[SPIIR_MAX_DET], W[SPIIR_MAX_DET], woff[SPIIR_MAX_DET];   // window of detector I vs T: first delta, width, row offset
  int32_t win_rows;                                           // total rows
  int32_t win_elems;                                          // float2 elements of the window region (even)
  spiir_sky_result* out; float* map;
};

struct PairInfo { int32_t slot, slide, valid, row; float2 vT; long long k; };

__device__ __forceinline__ int unpack_delta(const int32_t w1, const int32_t w2, int I) {
  if (I == 0) return 0;
  if (I == 1) return (int)(short)(w1 & 0xFFFF);
  if (I == 2) return (int)(short)((unsigned)w1 >> 16);
  return w2;
}

template <int D, bool MAP>
__global__ void __launch_bounds__(kSkyThreads, 2) k_sky(const __grid_constant__ SkyParams P) {
  constexpr int NQ = SkyRec<D>::NQ, RW = SkyRec<D>::RW;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* win = reinterpret_cast<float2*>(smem_raw);                              // [win_rows][NPS]
  float* tiles = reinterpret_cast<float*>(win + P.win_elems);                     // [warps][32][RW]
  float* red_c = tiles + kSkyWarps * 32 * RW;                                     // [warps][NP]
  int* red_p = reinterpret_cast<int*>(red_c + kSkyWarps * kSkyNP);                // [warps][NP]
  PairInfo* pinfo = reinterpret_cast<PairInfo*>(red_p + kSkyWarps * kSkyNP);      // [NP]

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int T = P.T;
  const int S1 = P.n_slides > 0 ? P.n_slides : 1;
  const long long n_pairs = (long long)P.counts[T] * S1;
  const long long n_batches = (n_pairs + kSkyNP - 1) / kSkyNP;
  const int64_t kmin = (P.k_newest - P.ring_len + 1 > 0) ? P.k_newest - P.ring_len + 1 : 0;
  float* mytile = tiles + warp * 32 * RW;
  const int rbeg = min(P.n_rec, warp * P.rec_per_warp), rend = min(P.n_rec, rbeg + P.rec_per_warp);

  for (long long batch = blockIdx.x; batch < n_batches; batch += gridDim.x) {
    __syncthreads();                                   // previous batch fully consumed
    // ---- pair set-up: which trigger, which slide, is every gather inside the view
    if (tid < kSkyNP) {
      PairInfo pi; pi.slot = -1; pi.slide = 0; pi.valid = 0; pi.row = 0; pi.vT = make_float2(0.f, 0.f); pi.k = 0;
      const long long q = batch * kSkyNP + tid;
      if (q < n_pairs) {
        pi.slot = P.list[q / S1];
        pi.slide = (int)(q % S1) + (P.n_slides > 0 ? 1 : 0);
        const spiir_trigger tr = P.trig[pi.slot];
        pi.row = tr.tmpl; pi.k = tr.k;
        bool ok = tr.k >= kmin && tr.k <= P.k_newest;
#pragma unroll
        for (int I = 0; I < D; ++I) {
          if (I == T) continue;
          const int64_t k0 = tr.k - (int64_t)pi.slide * P.step * P.mult[I] + P.lo[I];
          ok = ok && k0 >= kmin && k0 + P.W[I] - 1 <= P.k_newest;
        }
        pi.valid = ok ? 1 : 0;
        if (ok) pi.vT = P.z[(size_t)T * P.det_stride + (size_t)tr.tmpl * P.row_stride + (size_t)(tr.k % P.ring_len)];
      }
      pinfo[tid] = pi;
    }
    __syncthreads();
    // ---- delay windows -> shared memory, [row][pair]; a warp reads 32 consecutive samples of one pair
#pragma unroll
    for (int I = 0; I < D; ++I) {
      if (I == T) continue;
      const int W = P.W[I];
      const int Wp = (W + 31) & ~31;
      float2* dst = win + (size_t)P.woff[I] * kSkyNPS;
      for (int idx = tid; idx < kSkyNP * Wp; idx += kSkyThreads) {
        const int j = idx / Wp, r = idx - j * Wp;
        if (r >= W) continue;
        const PairInfo pi = pinfo[j];
        float2 v = make_float2(0.f, 0.f);
        if (pi.valid) {
          const int64_t k0 = pi.k - (int64_t)pi.slide * P.step * P.mult[I] + P.lo[I] + r;
          v = P.z[(size_t)I * P.det_stride + (size_t)pi.row * P.row_stride + (size_t)(k0 % P.ring_len)];
        }
        dst[(size_t)r * kSkyNPS + j] = v;
      }
    }
    __syncthreads();

    // ---- the direction stream: this warp's share, tile by tile
    float2 vT[kSkyK];
    float best[kSkyK]; int bpix[kSkyK];
#pragma unroll
    for (int a = 0; a < kSkyK; ++a) { vT[a] = pinfo[lane + 32 * a].vT; best[a] = -1.f; bpix[a] = INT_MAX; }
    long long mrow[kSkyK];                                  // sky-map row of each pair, -1 = none
#pragma unroll
    for (int a = 0; a < kSkyK; ++a) {
      const PairInfo pi = pinfo[lane + 32 * a];
      mrow[a] = (MAP && pi.valid) ? (long long)pi.slot * P.n_pix : -1;
    }
    float q[kSkyK][NQ];
#pragma unroll
    for (int a = 0; a < kSkyK; ++a)
#pragma unroll
      for (int e = 0; e < NQ; ++e) q[a][e] = 0.f;
    int cur_w1 = INT_MIN, cur_w2 = INT_MIN;

    float4 pre[RW / 4];
    if (rbeg < rend) {
      const int r = min(rbeg + lane, P.n_rec - 1);
#pragma unroll
      for (int c = 0; c < RW / 4; ++c) pre[c] = __ldg(reinterpret_cast<const float4*>(P.rec + (size_t)r * RW) + c);
    }
    for (int t0 = rbeg; t0 < rend; t0 += 32) {
      __syncwarp();
#pragma unroll
      for (int c = 0; c < RW / 4; ++c) reinterpret_cast<float4*>(mytile + lane * RW)[c] = pre[c];
      __syncwarp();
      if (t0 + 32 < rend) {                                   // prefetch the next tile while this one is consumed
        const int r = min(t0 + 32 + lane, P.n_rec - 1);
#pragma unroll
        for (int c = 0; c < RW / 4; ++c) pre[c] = __ldg(reinterpret_cast<const float4*>(P.rec + (size_t)r * RW) + c);
      }
      const int cnt = min(32, rend - t0);
      for (int r = 0; r < cnt; ++r) {
        float w[RW];
#pragma unroll
        for (int c = 0; c < RW / 4; ++c) {
          const float4 v = reinterpret_cast<const float4*>(mytile + r * RW)[c];   // broadcast read
          w[4 * c] = v.x; w[4 * c + 1] = v.y; w[4 * c + 2] = v.z; w[4 * c + 3] = v.w;
        }
        const int pix = __float_as_int(w[NQ]);
        const int w1 = __float_as_int(w[NQ + 1]);
        const int w2 = (D > 3) ? __float_as_int(w[NQ + 2]) : 0;
        if (w1 != cur_w1 || w2 != cur_w2) {                   // new delay tuple: gather once, form q_IJ once
          cur_w1 = w1; cur_w2 = w2;
          const int dT = unpack_delta(w1, w2, T);
#pragma unroll
          for (int a = 0; a < kSkyK; ++a) {
            float2 v[D];
#pragma unroll
            for (int I = 0; I < D; ++I) {
              if (I == T) { v[I] = vT[a]; continue; }
              const int row = P.woff[I] + (unpack_delta(w1, w2, I) - dT - P.lo[I]);
              v[I] = win[(size_t)row * kSkyNPS + lane + 32 * a];
            }
#pragma unroll
            for (int I = 0; I < D; ++I) q[a][I] = fmaf(v[I].x, v[I].x, v[I].y * v[I].y);
            int e = D;
#pragma unroll
            for (int J = 1; J < D; ++J)
#pragma unroll
              for (int I = 0; I < J; ++I) { q[a][e] = fmaf(v[I].x, v[J].x, v[I].y * v[J].y); ++e; }
          }
        }
#pragma unroll
        for (int a = 0; a < kSkyK; ++a) {
          float c = w[0] * q[a][0];
#pragma unroll
          for (int e = 1; e < NQ; ++e) c = fmaf(w[e], q[a][e], c);
          if (MAP) {
            if (mrow[a] >= 0) P.map[mrow[a] + pix] = c;
          }
          if (c >= best[a]) {
            if (c > best[a] || pix < bpix[a]) { best[a] = c; bpix[a] = pix; }
          }
        }
      }
    }
#pragma unroll
    for (int a = 0; a < kSkyK; ++a) {
      red_c[warp * kSkyNP + lane + 32 * a] = best[a];
      red_p[warp * kSkyNP + lane + 32 * a] = bpix[a];
    }
    __syncthreads();
    // ---- across the warps, then tot2 / null2 at the winning direction (Eq. 10)
    if (tid < kSkyNP) {
      const PairInfo pi = pinfo[tid];
      if (pi.slot >= 0) {
        spiir_sky_result res; res.coh2 = 0.f; res.null2 = 0.f; res.tot2 = 0.f; res.pix = -1;
        if (pi.valid) {
          float bc = red_c[tid]; int bp = red_p[tid];
          for (int wv = 1; wv < kSkyWarps; ++wv) {
            const float c = red_c[wv * kSkyNP + tid]; const int p = red_p[wv * kSkyNP + tid];
            if (c > bc || (c == bc && p < bp)) { bc = c; bp = p; }
          }
          const int4 dl = __ldg(reinterpret_cast<const int4*>(P.pix_delta) + bp);
          const int dd[4] = {0, dl.y, dl.z, dl.w};
          float tot = 0.f;
#pragma unroll
          for (int I = 0; I < D; ++I) {
            float2 v;
            if (I == T) v = pi.vT;
            else v = win[(size_t)(P.woff[I] + (dd[I] - dd[T] - P.lo[I])) * kSkyNPS + tid];
            tot += fmaf(v.x, v.x, v.y * v.y);
          }
          res.coh2 = bc; res.tot2 = tot; res.null2 = fmaxf(tot - bc, 0.f); res.pix = bp;
        }
        P.out[(size_t)pi.slot * S1 + (P.n_slides > 0 ? pi.slide - 1 : 0)] = res;
      }
    }
  }
}

// valid slots -> per-detector lists; invalid slots get their "no result" rows here
__global__ void __launch_bounds__(256) k_sky_bin(const spiir_trigger* trig, int n_slots, int n_det, int S1,
                                                 int32_t* lists, int32_t* counts, int max_slots,
                                                 spiir_sky_result* out) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= n_slots) return;
  const spiir_trigger t = trig[i];
  if (t.valid && t.det >= 0 && t.det < n_det) {
    const int pos = atomicAdd(counts + t.det, 1);
    lists[(size_t)t.det * max_slots + pos] = i;
  } else {
    spiir_sky_result r; r.coh2 = 0.f; r.null2 = 0.f; r.tot2 = 0.f; r.pix = -1;
    for (int s = 0; s < S1; ++s) out[(size_t)i * S1 + s] = r;
  }
}

}  // namespace spiir

using namespace spiir;

struct spiir_sky_plan {
  int n_det = 0, n_pix = 0, max_slots = 0, n_rec = 0, n_tuples = 0, rec_per_warp = 0, RW = 0;
  char* ws = nullptr;
  size_t off_rec = 0, off_pixd = 0, off_lists = 0, off_counts = 0, bytes = 0;
  int lo[SPIIR_MAX_DET][SPIIR_MAX_DET], hi[SPIIR_MAX_DET][SPIIR_MAX_DET];    // [T][I]
  int num_sms = 148;
};

static size_t sky_align(size_t x) { return (x + 255) / 256 * 256; }
static int sky_win_elems(int rows) { return (rows * kSkyNPS + 1) & ~1; }
static size_t sky_smem_bytes(int rows, int RW) {
  return (size_t)sky_win_elems(rows) * 8 + (size_t)kSkyWarps * 32 * RW * 4 + (size_t)kSkyWarps * kSkyNP * 8 +
         kSkyNP * sizeof(PairInfo);
}

static void sky_layout(spiir_sky_plan* pl) {
  const int D = pl->n_det;
  pl->RW = (D * (D + 1) / 2 + 3 + 3) / 4 * 4;
  size_t cur = 0;
  pl->off_rec = cur;    cur = sky_align(cur + (size_t)pl->n_pix * pl->RW * 4);
  pl->off_pixd = cur;   cur = sky_align(cur + (size_t)pl->n_pix * 16);
  pl->off_lists = cur;  cur = sky_align(cur + (size_t)D * pl->max_slots * 4);
  pl->off_counts = cur; cur = sky_align(cur + SPIIR_MAX_DET * 4);
  pl->bytes = cur;
}

extern "C" {

int spiir_sky_plan_workspace_bytes(int32_t n_det, int32_t n_pix, int32_t max_slots, size_t* bytes) {
  SPIIR_REQUIRE(n_det >= 2 && n_det <= SPIIR_MAX_DET, "n_det %d out of range", n_det);
  SPIIR_REQUIRE(n_pix >= 1 && max_slots >= 1 && bytes, "bad n_pix / max_slots / bytes");
  spiir_sky_plan pl; pl.n_det = n_det; pl.n_pix = n_pix; pl.max_slots = max_slots;
  sky_layout(&pl);
  *bytes = pl.bytes;
  return SPIIR_OK;
}

int spiir_sky_plan_init(spiir_sky_plan** out, int32_t n_det, int32_t n_pix, int32_t max_slots, const float* u2,
                        const int32_t* delay, void* dev_workspace, size_t bytes, void* stream) {
  SPIIR_REQUIRE(out && u2 && delay && dev_workspace, "a pointer is NULL");
  SPIIR_REQUIRE(n_det >= 2 && n_det <= SPIIR_MAX_DET, "n_det %d out of range", n_det);
  SPIIR_REQUIRE(n_pix >= 1 && max_slots >= 1, "bad n_pix / max_slots");
  SPIIR_REQUIRE(((uintptr_t)dev_workspace & 255) == 0, "workspace must be 256-byte aligned");
  spiir_sky_plan* pl = new spiir_sky_plan();
  pl->n_det = n_det; pl->n_pix = n_pix; pl->max_slots = max_slots;
  sky_layout(pl);
  if (bytes < pl->bytes) { set_error("workspace too small: %zu < %zu", bytes, pl->bytes); delete pl; return SPIIR_ENOMEM; }
  const int D = n_det, NQ = D * (D + 1) / 2, RW = pl->RW;
  for (int T = 0; T < D; ++T) for (int I = 0; I < D; ++I) { pl->lo[T][I] = INT_MAX; pl->hi[T][I] = INT_MIN; }
  std::vector<int32_t> pixd((size_t)n_pix * 4, 0);
  for (int p = 0; p < n_pix; ++p) {
    for (int I = 0; I < D; ++I) {
      const long long d = (long long)delay[(size_t)p * D + I] - delay[(size_t)p * D];
      if (d < -32000 || d > 32000) { set_error("pixel %d: delay difference %lld does not fit the plan", p, d); delete pl; return SPIIR_EINVAL; }
      pixd[(size_t)p * 4 + I] = (int32_t)d;
    }
    for (int T = 0; T < D; ++T) for (int I = 0; I < D; ++I) {
      const int d = delay[(size_t)p * D + I] - delay[(size_t)p * D + T];
      pl->lo[T][I] = std::min(pl->lo[T][I], d); pl->hi[T][I] = std::max(pl->hi[T][I], d);
    }
  }
  // directions sorted by delay tuple, then by pixel index
  std::vector<int32_t> order(n_pix);
  for (int p = 0; p < n_pix; ++p) order[p] = p;
  std::sort(order.begin(), order.end(), [&](int32_t x, int32_t y) {
    for (int I = 1; I < D; ++I) {
      const int32_t dx = pixd[(size_t)x * 4 + I], dy = pixd[(size_t)y * 4 + I];
      if (dx != dy) return dx < dy;
    }
    return x < y;
  });
  std::vector<float> rec((size_t)n_pix * RW, 0.f);
  int n_tuples = 0;
  for (int r = 0; r < n_pix; ++r) {
    const int p = order[r];
    float* w = rec.data() + (size_t)r * RW;
    const float* u = u2 + (size_t)p * D * 2;
    // projector M = U2 U2^T in float64 from the float32 table, rounded once
    for (int I = 0; I < D; ++I) w[I] = (float)((double)u[2 * I] * u[2 * I] + (double)u[2 * I + 1] * u[2 * I + 1]);
    int e = D;
    for (int J = 1; J < D; ++J)
      for (int I = 0; I < J; ++I)
        w[e++] = (float)(2.0 * ((double)u[2 * I] * u[2 * J] + (double)u[2 * I + 1] * u[2 * J + 1]));
    int32_t iw[3];
    iw[0] = p;
    iw[1] = (int32_t)(((uint32_t)(uint16_t)(int16_t)pixd[(size_t)p * 4 + 1]) |
                      ((uint32_t)(uint16_t)(int16_t)(D > 2 ? pixd[(size_t)p * 4 + 2] : 0) << 16));
    iw[2] = D > 3 ? pixd[(size_t)p * 4 + 3] : 0;
    memcpy(w + NQ, iw, sizeof(iw));
    if (r == 0 || memcmp(&pixd[(size_t)p * 4], &pixd[(size_t)order[r - 1] * 4], 16) != 0) ++n_tuples;
  }
  pl->n_rec = n_pix; pl->n_tuples = n_tuples;
  pl->rec_per_warp = ((n_pix + kSkyWarps - 1) / kSkyWarps + 31) / 32 * 32;
  // shared-memory need of the widest trigger detector
  for (int T = 0; T < D; ++T) {
    int rows = 0;
    for (int I = 0; I < D; ++I) if (I != T) rows += pl->hi[T][I] - pl->lo[T][I] + 1;
    const size_t smem = sky_smem_bytes(rows, RW);
    if (smem > (size_t)kSkySmemMax) {
      set_error("delay span of trigger detector %d needs %zu bytes of shared memory (> %d)", T, smem, kSkySmemMax);
      delete pl; return SPIIR_EINVAL;
    }
  }
  pl->ws = (char*)dev_workspace;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemcpyAsync(pl->ws + pl->off_rec, rec.data(), rec.size() * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(pl->ws + pl->off_pixd, pixd.data(), pixd.size() * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  int dev = 0, sms = 0;
  if (e == cudaSuccess) e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) { set_error("sky plan upload failed: %s", cudaGetErrorString(e)); delete pl; return SPIIR_ECUDA; }
  pl->num_sms = sms > 0 ? sms : 148;
  *out = pl;
  return SPIIR_OK;
}

int spiir_sky_plan_free(spiir_sky_plan* pl) {
  SPIIR_REQUIRE(pl != nullptr, "plan is NULL");
  delete pl;
  return SPIIR_OK;
}

int32_t spiir_sky_plan_tuples(const spiir_sky_plan* pl) { return pl ? pl->n_tuples : 0; }

}  // extern "C"

template <int D, bool MAP>
static int sky_launch_one(const SkyParams& P, int grid, size_t smem, cudaStream_t st) {
  static size_t configured = 0;
  if (smem > configured) {
    SPIIR_CUDA_OK(cudaFuncSetAttribute(k_sky<D, MAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSkySmemMax));
    configured = kSkySmemMax;
  }
  k_sky<D, MAP><<<grid, kSkyThreads, smem, st>>>(P);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

static int sky_run(spiir_sky_plan* pl, const spiir_snr_view* view, const spiir_trigger* trig, int32_t n_slots,
                   int32_t n_slides, int64_t step, const int32_t* mult, spiir_sky_result* out, float* map,
                   cudaStream_t st) {
  SPIIR_REQUIRE(pl && view && trig && out, "a pointer is NULL");
  SPIIR_REQUIRE(view->dev_z && view->ring_len >= 1, "bad SNR view");
  SPIIR_REQUIRE(n_slots >= 0 && n_slots <= pl->max_slots, "n_slots %d exceeds the plan's max_slots %d", n_slots,
                pl->max_slots);
  SPIIR_REQUIRE(n_slides >= 0, "n_slides < 0");
  SPIIR_REQUIRE(n_slides == 0 || (mult != nullptr && step >= 0), "time slides need host_slide_mult and step >= 0");
  if (n_slots == 0) return SPIIR_OK;
  const int D = pl->n_det, S1 = n_slides > 0 ? n_slides : 1;
  int32_t* counts = (int32_t*)(pl->ws + pl->off_counts);
  int32_t* lists = (int32_t*)(pl->ws + pl->off_lists);
  SPIIR_CUDA_OK(cudaMemsetAsync(counts, 0, SPIIR_MAX_DET * 4, st));
  if (map) SPIIR_CUDA_OK(cudaMemsetAsync(map, 0, (size_t)n_slots * pl->n_pix * sizeof(float), st));
  k_sky_bin<<<(n_slots + 255) / 256, 256, 0, st>>>(trig, n_slots, D, S1, lists, counts, pl->max_slots, out);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  for (int T = 0; T < D; ++T) {
    SkyParams P;
    memset(&P, 0, sizeof(P));
    P.rec = (const float*)(pl->ws + pl->off_rec); P.n_rec = pl->n_rec; P.rec_per_warp = pl->rec_per_warp;
    P.pix_delta = (const int32_t*)(pl->ws + pl->off_pixd); P.n_pix = pl->n_pix;
    P.z = (const float2*)view->dev_z; P.det_stride = view->det_stride; P.row_stride = view->row_stride;
    P.ring_len = view->ring_len; P.k_newest = view->k_newest;
    P.trig = trig; P.list = lists + (size_t)T * pl->max_slots; P.counts = counts; P.T = T;
    P.n_slides = n_slides; P.step = step;
    int rows = 0;
    for (int I = 0; I < D; ++I) {
      P.mult[I] = (mult && I != T) ? mult[I] : 0;
      P.lo[I] = pl->lo[T][I]; P.W[I] = pl->hi[T][I] - pl->lo[T][I] + 1;
      P.woff[I] = rows;
      if (I != T) rows += P.W[I];
    }
    P.win_rows = rows; P.win_elems = sky_win_elems(rows);
    P.out = out; P.map = map;
    const size_t smem = sky_smem_bytes(rows, pl->RW);
    const long long max_batches = ((long long)n_slots * S1 + kSkyNP - 1) / kSkyNP;
    const int grid = (int)std::min<long long>(max_batches, (long long)pl->num_sms * 2);
    int rc;
    if (D == 2)      rc = map ? sky_launch_one<2, true>(P, grid, smem, st) : sky_launch_one<2, false>(P, grid, smem, st);
    else if (D == 3) rc = map ? sky_launch_one<3, true>(P, grid, smem, st) : sky_launch_one<3, false>(P, grid, smem, st);
    else             rc = map ? sky_launch_one<4, true>(P, grid, smem, st) : sky_launch_one<4, false>(P, grid, smem, st);
    if (rc) return rc;
  }
  return SPIIR_OK;
}

extern "C" {

int coherent_sky_search(spiir_sky_plan* plan, const spiir_snr_view* view, const spiir_trigger* dev_trig,
                        int32_t n_slots, spiir_sky_result* dev_out, float* dev_skymap, void* stream) {
  return sky_run(plan, view, dev_trig, n_slots, 0, 0, nullptr, dev_out, dev_skymap, (cudaStream_t)stream);
}

int timeslide_background(spiir_sky_plan* bg_plan, const spiir_snr_view* view, const spiir_trigger* dev_trig,
                         int32_t n_slots, int32_t n_slides, int64_t step_samples, const int32_t* host_slide_mult,
                         spiir_sky_result* dev_out, void* stream) {
  SPIIR_REQUIRE(n_slides >= 1, "n_slides must be >= 1");
  return sky_run(bg_plan, view, dev_trig, n_slots, n_slides, step_samples, host_slide_mult, dev_out, nullptr,
                 (cudaStream_t)stream);
}

}  // extern "C"
