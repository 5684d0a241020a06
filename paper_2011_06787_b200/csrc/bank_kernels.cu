// Device kernels of the SPIIR filter bank (H0-H3 of DESIGN.md) for sm_100a.
//
//   k_prep    H0  history shift + x2 decimator chain + 4 pre-shifted replicas per band
//   k_bank    H1+H2 delay fetch + IIR recursion + per-unit band sums (THE hot loop); the band above the
//             output rate advances two samples per step (a^2, a b precomputed)
//   k_combine H3  unit sums -> band sums -> interpolating cascade -> SNR ring, fused
//                 per-template peak tracking (H4 mode 0)
//
// PAPER.md:129 (Eq. 8): y_l[k] = a_l y_l[k-1] + b_l x[k-d_l]; z[k] = sum_l y_l[k];
// templates and filters are independent -> GPU threads.  The mapping,
// the replica trick and the reduction are this implementation's own.
#include "spiir_internal.cuh"

namespace spiir {

// ---------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
// Bounded wait: try_wait suspends the thread for a hardware time slice per poll; a copy that faulted or an
// expect_tx that disagrees with the bytes issued traps after seconds instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
#pragma unroll 1
  for (uint32_t spin = 0; spin < (1u << 26); ++spin) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (done) return;
  }
  __trap();
}
// 1-D TMA bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ------------------------------------------------------------------- k_prep

constexpr int kPrepThreads = 512;
constexpr int kPrepStage = 4096 + 32;

__global__ void __launch_bounds__(kPrepThreads) k_prep(PrepParams p) {
  __shared__ __align__(16) float stage[kPrepStage];
  __shared__ float g[SPIIR_FIR_TAPS];
  const int det = blockIdx.x, tid = threadIdx.x;
  if (tid < SPIIR_FIR_TAPS) g[tid] = p.taps_dec[tid];
  for (int b = 0; b < p.n_bands; ++b) {
    float* xn = p.xnew[b] + det * p.x_det_stride[b];
    const float* xo = p.xold[b] + det * p.x_det_stride[b];
    const int H = p.Hcap[b], n = p.n[b], pn = p.prev_n[b], cap = p.cap[b];
    // (a) carry the last H samples of the previous layout to the front of the new one
    for (int j = tid; j < H; j += kPrepThreads) xn[j] = xo[pn + j];
    // (b) the new samples of this band
    if (b == 0) {
      const float4* src = reinterpret_cast<const float4*>(p.strain + (size_t)det * p.n0);
      float4* dst = reinterpret_cast<float4*>(xn + H);
      for (int j = tid; j < n / 4; j += kPrepThreads) dst[j] = __ldg(src + j);   // coalesced float4 loads
    } else {
      // x_b[m] = sum_j g[j] x_{b-1}[2m+1-j]: stage band b-1 (31 samples of history + its new
      // samples) in shared memory with float4 loads, then every thread forms outputs.
      const float* xp = p.xnew[b - 1] + det * p.x_det_stride[b - 1] + p.Hcap[b - 1] - 32;
      const int np = p.n[b - 1] + 32;
      __syncthreads();                       // band b-1 complete, previous use of stage[] finished
      for (int j = tid; j < np / 4; j += kPrepThreads)
        reinterpret_cast<float4*>(stage)[j] = reinterpret_cast<const float4*>(xp)[j];
      __syncthreads();
      for (int m = tid; m < n; m += kPrepThreads) {
        float acc = 0.f;
#pragma unroll
        for (int j = 0; j < SPIIR_FIR_TAPS; ++j) acc = fmaf(g[j], stage[32 + 2 * m + 1 - j], acc);
        xn[H + m] = acc;
      }
    }
    __syncthreads();
    // (c) replicas r = 1..nrep-1: rep_r[j] = rep_0[j + r]  (aligned float4 reads for any delay)
    const int tot = H + n, nrep = p.nrep[b];
    for (int j = tid; j < tot; j += kPrepThreads) {
      for (int r = 1; r < nrep; ++r) xn[(size_t)r * cap + j] = (j + r < tot) ? xn[j + r] : 0.f;
    }
  }
}

void launch_prep(const PrepParams& p, int n_det, cudaStream_t st) {
  k_prep<<<n_det, kPrepThreads, 0, st>>>(p);
  count_launch();
}

// ------------------------------------------------------------------- k_bank
// Sum 8 per-lane values (4 complex samples) over the G lanes of a unit.  After the
// three halving steps lane (g & 7) holds element (g & 7) summed over its 8-lane
// group; wider units finish with plain butterflies.
template <int G>
__device__ __forceinline__ float reduce8(float (&s)[8], int lane) {
  float w[4], u[2], t;
  const bool b4 = lane & 4, b2 = lane & 2, b1 = lane & 1;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const float send = b4 ? s[j] : s[j + 4];
    const float keep = b4 ? s[j + 4] : s[j];
    w[j] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const float send = b2 ? w[j] : w[j + 2];
    const float keep = b2 ? w[j + 2] : w[j];
    u[j] = keep + __shfl_xor_sync(0xffffffffu, send, 2);
  }
  {
    const float send = b1 ? u[0] : u[1];
    const float keep = b1 ? u[1] : u[0];
    t = keep + __shfl_xor_sync(0xffffffffu, send, 1);
  }
  if (G >= 16) t += __shfl_xor_sync(0xffffffffu, t, 8);
  if (G >= 32) t += __shfl_xor_sync(0xffffffffu, t, 16);
  return t;
}

// Same for 4 per-lane values (2 complex samples): after two halving steps and one
// butterfly lanes g and g^1 both hold element (g >> 1) & 3 summed over their 8-lane group.
template <int G>
__device__ __forceinline__ float reduce4(float (&s)[4], int lane) {
  float w[2], u, t;
  const bool b4 = lane & 4, b2 = lane & 2;
#pragma unroll
  for (int j = 0; j < 2; ++j) {
    const float send = b4 ? s[j] : s[j + 2];
    const float keep = b4 ? s[j + 2] : s[j];
    w[j] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  {
    const float send = b2 ? w[0] : w[1];
    const float keep = b2 ? w[1] : w[0];
    u = keep + __shfl_xor_sync(0xffffffffu, send, 2);
  }
  t = u + __shfl_xor_sync(0xffffffffu, u, 1);
  if (G >= 16) t += __shfl_xor_sync(0xffffffffu, t, 8);
  if (G >= 32) t += __shfl_xor_sync(0xffffffffu, t, 16);
  return t;
}

template <int F>
struct FilterRegs {
  float ar[F], ai[F], br[F], bi[F], yr[F], yi[F];   // in a two-sample (odd-only) band ar/ai hold a^2
  float abr[F], abi[F];                             // a b, two-sample bands only (dead otherwise)
  int off[F];
};

// Four consecutive samples of all F filters of this lane; s[] receives the lane's
// partial sums (re0, im0, re1, im1, ...).  Per update: FMUL + 2 FFMA per component
// and one FADD per component into the sum = 8 FP32 lane-operations (12 flop,
// PAPER.md:135).  Filters are taken two at a time so that the FFMAs and FADDs issue
// as packed FFMA2 / FADD2 (sm_100 f32x2: same FP32-pipe cycles, half the issue
// slots): per two updates 4 FMUL + 4 FFMA2 + 2 FADD2.  An odd last filter runs scalar.
// ODD: only samples 1 and 3 of the four enter a sum (a band running at twice the output
// rate contributes z[m] += s_0[2m+1] only, reading M5); s[] = (re1, im1, re3, im3).
template <int F, bool XG, bool ODD>
__device__ __forceinline__ void step4(FilterRegs<F>& r, const float* __restrict__ x, int i, float (&s)[ODD ? 4 : 8]) {
  float2 sr[4], si[4];                       // (sum over even filters, sum over odd filters)
#pragma unroll
  for (int f = 0; f + 1 < F; f += 2) {
    float4 xa, xb;
    if (XG) {
      xa = __ldg(reinterpret_cast<const float4*>(x + r.off[f] + i));
      xb = __ldg(reinterpret_cast<const float4*>(x + r.off[f + 1] + i));
    } else {
      xa = *reinterpret_cast<const float4*>(x + r.off[f] + i);
      xb = *reinterpret_cast<const float4*>(x + r.off[f + 1] + i);
    }
    const float xsa[4] = {xa.x, xa.y, xa.z, xa.w}, xsb[4] = {xb.x, xb.y, xb.z, xb.w};
    const float2 ar = make_float2(r.ar[f], r.ar[f + 1]), ai = make_float2(r.ai[f], r.ai[f + 1]);
    const float2 nai = make_float2(-r.ai[f], -r.ai[f + 1]);
    float2 yr = make_float2(r.yr[f], r.yr[f + 1]), yi = make_float2(r.yi[f], r.yi[f + 1]);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float2 pr = make_float2(r.br[f] * xsa[q], r.br[f + 1] * xsb[q]);
      const float2 pi = make_float2(r.bi[f] * xsa[q], r.bi[f + 1] * xsb[q]);
      const float2 tr = __ffma2_rn(nai, yi, pr);
      const float2 ti = __ffma2_rn(ai, yr, pi);
      const float2 nr = __ffma2_rn(ar, yr, tr);
      const float2 ni = __ffma2_rn(ar, yi, ti);
      yr = nr; yi = ni;
      if (!ODD || (q & 1)) {
        if (f == 0) { sr[q] = yr; si[q] = yi; }
        else        { sr[q] = __fadd2_rn(sr[q], yr); si[q] = __fadd2_rn(si[q], yi); }
      }
    }
    r.yr[f] = yr.x; r.yr[f + 1] = yr.y; r.yi[f] = yi.x; r.yi[f + 1] = yi.y;
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (ODD && !(q & 1)) continue;
    const int o = ODD ? (q >> 1) : q;
    s[2 * o] = (F > 1) ? sr[q].x + sr[q].y : 0.f;
    s[2 * o + 1] = (F > 1) ? si[q].x + si[q].y : 0.f;
  }
  if (F & 1) {
    constexpr int f = F - 1;
    float4 xv;
    if (XG) xv = __ldg(reinterpret_cast<const float4*>(x + r.off[f] + i));
    else    xv = *reinterpret_cast<const float4*>(x + r.off[f] + i);
    const float xs[4] = {xv.x, xv.y, xv.z, xv.w};
    float yr = r.yr[f], yi = r.yi[f];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float tr = fmaf(-r.ai[f], yi, r.br[f] * xs[q]);
      const float ti = fmaf(r.ai[f], yr, r.bi[f] * xs[q]);
      const float nr = fmaf(r.ar[f], yr, tr);
      const float ni = fmaf(r.ar[f], yi, ti);
      yr = nr; yi = ni;
      if (!ODD || (q & 1)) {
        const int o = ODD ? (q >> 1) : q;
        s[2 * o] += yr; s[2 * o + 1] += yi;
      }
    }
    r.yr[f] = yr; r.yi[f] = yi;
  }
}

// The band above the output rate contributes its odd samples only (reading M5), so its recursion advances TWO
// samples per step - north_star's "chunked scan using precomputed a1 powers", chunk = 2:
//   y[2m+1] = a^2 y[2m-1] + (a b) x[2m-d] + b x[2m+1-d]
// with a^2 and a b formed in float64 at init: 8 multiply-adds + 2 adds per two filter-samples instead of 12 + 2.
// Four input samples = two steps; s[] = (re1, im1, re3, im3).  Pairs of filters packed as in step4.
template <int F, bool XG>
__device__ __forceinline__ void step2x2(FilterRegs<F>& r, const float* __restrict__ x, int i, float (&s)[4]) {
  float2 sr[2], si[2];
#pragma unroll
  for (int f = 0; f + 1 < F; f += 2) {
    float4 xa, xb;
    if (XG) {
      xa = __ldg(reinterpret_cast<const float4*>(x + r.off[f] + i));
      xb = __ldg(reinterpret_cast<const float4*>(x + r.off[f + 1] + i));
    } else {
      xa = *reinterpret_cast<const float4*>(x + r.off[f] + i);
      xb = *reinterpret_cast<const float4*>(x + r.off[f + 1] + i);
    }
    const float xsa[4] = {xa.x, xa.y, xa.z, xa.w}, xsb[4] = {xb.x, xb.y, xb.z, xb.w};
    const float2 a2r = make_float2(r.ar[f], r.ar[f + 1]), a2i = make_float2(r.ai[f], r.ai[f + 1]);
    const float2 na2i = make_float2(-r.ai[f], -r.ai[f + 1]);
    float2 yr = make_float2(r.yr[f], r.yr[f + 1]), yi = make_float2(r.yi[f], r.yi[f + 1]);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float2 pr = make_float2(fmaf(r.abr[f], xsa[2 * h], r.br[f] * xsa[2 * h + 1]),
                                    fmaf(r.abr[f + 1], xsb[2 * h], r.br[f + 1] * xsb[2 * h + 1]));
      const float2 pi = make_float2(fmaf(r.abi[f], xsa[2 * h], r.bi[f] * xsa[2 * h + 1]),
                                    fmaf(r.abi[f + 1], xsb[2 * h], r.bi[f + 1] * xsb[2 * h + 1]));
      const float2 tr = __ffma2_rn(na2i, yi, pr);
      const float2 ti = __ffma2_rn(a2i, yr, pi);
      const float2 nr = __ffma2_rn(a2r, yr, tr);
      const float2 ni = __ffma2_rn(a2r, yi, ti);
      yr = nr; yi = ni;
      if (f == 0) { sr[h] = yr; si[h] = yi; }
      else        { sr[h] = __fadd2_rn(sr[h], yr); si[h] = __fadd2_rn(si[h], yi); }
    }
    r.yr[f] = yr.x; r.yr[f + 1] = yr.y; r.yi[f] = yi.x; r.yi[f + 1] = yi.y;
  }
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    s[2 * h] = (F > 1) ? sr[h].x + sr[h].y : 0.f;
    s[2 * h + 1] = (F > 1) ? si[h].x + si[h].y : 0.f;
  }
  if (F & 1) {
    constexpr int f = F - 1;
    float4 xv;
    if (XG) xv = __ldg(reinterpret_cast<const float4*>(x + r.off[f] + i));
    else    xv = *reinterpret_cast<const float4*>(x + r.off[f] + i);
    const float xs[4] = {xv.x, xv.y, xv.z, xv.w};
    float yr = r.yr[f], yi = r.yi[f];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const float pr = fmaf(r.abr[f], xs[2 * h], r.br[f] * xs[2 * h + 1]);
      const float pi = fmaf(r.abi[f], xs[2 * h], r.bi[f] * xs[2 * h + 1]);
      const float nr = fmaf(r.ar[f], yr, fmaf(-r.ai[f], yi, pr));
      const float ni = fmaf(r.ar[f], yi, fmaf(r.ai[f], yr, pi));
      yr = nr; yi = ni;
      s[2 * h] += yr; s[2 * h + 1] += yi;
    }
    r.yr[f] = yr; r.yi[f] = yi;
  }
}

// One sub-chunk of `len` samples for this lane's filters: recursion, unit sums, store.
template <int G, int F, bool XG, bool ODD>
__device__ __forceinline__ void run_samples(FilterRegs<F>& r, const float* __restrict__ x, int len, float* __restrict__ So,
                                            int lane, int g) {
  for (int i = 0; i < len; i += 4) {
    if (ODD) {
      float s[4];
      step2x2<F, XG>(r, x, i, s);
      const float t = reduce4<G>(s, lane);
      if (g < 8 && !(g & 1)) So[i + (g >> 1)] = t;          // 2 complex samples per 4 inputs
    } else {
      float s[8];
      step4<F, XG, false>(r, x, i, s);
      const float t = reduce8<G>(s, lane);
      if (g < 8) So[2 * i + g] = t;
    }
  }
}

template <int G, int F, bool ODD>
__global__ void __launch_bounds__(kBankThreads, 2)
k_bank(const __grid_constant__ BankParams P, const CtaWork* __restrict__ work) {
  extern __shared__ __align__(128) float xs[];
  // (Tried in round 2: the detector varying fastest over the grid, so that the three CTAs sharing a work item's
  // coefficients run side by side: DRAM reads of the two launches fell from 1.24 to 0.66 GB, the time ROSE by 1.7 %
  // (11.95 against 11.75 ms): the kernel is not HBM-bound and the order below keeps one detector's input in flight.)
  const CtaWork w = work[blockIdx.x];
  const BandDev& B = P.band[w.band];
  const int det = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wu = w.wu_begin + warp;
  const bool active = wu < w.wu_end;

  FilterRegs<F> r;
  const size_t slot0 = ((size_t)wu * F) * 32 + lane;
  float2* st = B.state + (size_t)det * B.state_det_stride;
  if (active) {
#pragma unroll
    for (int f = 0; f < F; ++f) {
      const float4 c = __ldg(B.coef + slot0 + f * 32);
      r.ar[f] = c.x; r.ai[f] = c.y; r.br[f] = c.z; r.bi[f] = c.w;
      r.off[f] = __ldg(B.off + slot0 + f * 32);
      if (ODD) { const float2 ab = __ldg(B.coef2 + slot0 + f * 32); r.abr[f] = ab.x; r.abi[f] = ab.y; }
      const float2 y = st[slot0 + f * 32];
      r.yr[f] = y.x; r.yi[f] = y.y;
    }
  }
  constexpr int UPW = 32 / G;                        // units per warp
  const int unit = wu * UPW + lane / G;
  const int g = lane % G;
  float* Sout = reinterpret_cast<float*>(B.S + (size_t)det * B.S_det_stride + (size_t)unit * B.nmax);
  const int n = B.n;

  if (w.xg) {
    // long-delay units (same launch, listed first): the replicas are read straight from
    // global memory (L1/L2 resident)
    if (active) {
      const float* x = B.xrep + (size_t)det * B.x_det_stride;
      run_samples<G, F, true, ODD>(r, x, n, Sout, lane, g);
    }
  } else {
    uint64_t* bar = reinterpret_cast<uint64_t*>(xs + B.nrep * B.reps);
    if (threadIdx.x == 0) mbar_init(bar, 1);
    __syncthreads();
    uint32_t phase = 0;
    const float* src0 = B.xrep + (size_t)det * B.x_det_stride + (B.Hcap - B.Hs - B.pad);
    for (int m0 = 0; m0 < n; m0 += B.nsub) {
      const int len = min(B.nsub, n - m0);
      if (m0 > 0) __syncthreads();                   // every warp finished reading the previous window
      if (threadIdx.x == 0) {
        const uint32_t bytes = (uint32_t)(B.pad + B.Hs + len) * 4u;
        mbar_expect_tx(bar, bytes * B.nrep);
        for (int rep = 0; rep < B.nrep; ++rep)
          tma_load_1d(xs + rep * B.reps, src0 + (size_t)rep * B.cap + m0, bytes, bar);
      }
      mbar_wait(bar, phase);
      phase ^= 1u;
      if (active) {
        run_samples<G, F, false, ODD>(r, xs, len, Sout + (ODD ? m0 : 2 * m0), lane, g);
      }
    }
  }
  if (active) {
#pragma unroll
    for (int f = 0; f < F; ++f) st[slot0 + f * 32] = make_float2(r.yr[f], r.yi[f]);
  }
}

template <int G, int F, bool ODD>
static int launch_one(const BankParams& P, const CtaWork* dev_work, int n_cta, int n_det, int smem, cudaStream_t st) {
  static unsigned long long configured = 0;
  if (first_use_on_device(configured)) {
    SPIIR_CUDA_OK(cudaFuncSetAttribute(k_bank<G, F, ODD>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  }
  k_bank<G, F, ODD><<<dim3(n_cta, n_det), kBankThreads, smem, st>>>(P, dev_work);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

#define SPIIR_F_CASES(G)                                                          \
  switch (F) {                                                                    \
    case 4:  return odd ? launch_one<G, 4, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 4, false>(P, dev_work, n_cta, n_det, smem, st);        \
    case 5:  return odd ? launch_one<G, 5, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 5, false>(P, dev_work, n_cta, n_det, smem, st);        \
    case 6:  return odd ? launch_one<G, 6, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 6, false>(P, dev_work, n_cta, n_det, smem, st);        \
    case 7:  return odd ? launch_one<G, 7, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 7, false>(P, dev_work, n_cta, n_det, smem, st);        \
    case 8:  return odd ? launch_one<G, 8, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 8, false>(P, dev_work, n_cta, n_det, smem, st);        \
    case 9:  return odd ? launch_one<G, 9, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 9, false>(P, dev_work, n_cta, n_det, smem, st);        \
    case 10: return odd ? launch_one<G, 10, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 10, false>(P, dev_work, n_cta, n_det, smem, st);       \
    case 11: return odd ? launch_one<G, 11, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 11, false>(P, dev_work, n_cta, n_det, smem, st);       \
    case 12: return odd ? launch_one<G, 12, true>(P, dev_work, n_cta, n_det, smem, st) : launch_one<G, 12, false>(P, dev_work, n_cta, n_det, smem, st);       \
    default: break;                                                               \
  }

int launch_bank_group(int G, int F, int odd, const BankParams& P, const CtaWork* dev_work, int n_cta, int n_det,
                      int smem, cudaStream_t st) {
  if (G == 8) { SPIIR_F_CASES(8) }
  else if (G == 16) { SPIIR_F_CASES(16) }
  else if (G == 32) { SPIIR_F_CASES(32) }
  set_error("no kernel instance for G=%d F=%d", G, F);
  return SPIIR_EINVAL;
}

// ---------------------------------------------------------------- k_combine

constexpr int kCombineThreads = 256;

__device__ __forceinline__ float2 unit_sum(const float2* __restrict__ S, int nmax, int first, int count, int m) {
  float2 a = make_float2(0.f, 0.f);
  for (int u = 0; u < count; ++u) {
    const float2 v = S[(size_t)(first + u) * nmax + m];
    a.x += v.x; a.y += v.y;
  }
  return a;
}

__device__ __forceinline__ void cp_async_16(void* dst_smem, const void* src_gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}

__global__ void __launch_bounds__(kCombineThreads) k_combine(const __grid_constant__ CombineParams p) {
  extern __shared__ __align__(16) float2 cbuf[];
  __shared__ float red_m2[kCombineThreads / 32];
  __shared__ int red_k[kCombineThreads / 32];
  const int t = blockIdx.x, det = blockIdx.y, tid = threadIdx.x;
  float hr[SPIIR_FIR_TAPS];                            // interpolation taps, in registers
#pragma unroll
  for (int j = 0; j < SPIIR_FIR_TAPS; ++j) hr[j] = __ldg(p.taps_int + j);
  float2* buf[2] = {cbuf, cbuf + p.bufA};              // bufA, bufB even: 16-byte aligned windows
  float2* sbuf = cbuf + ((p.bufA + p.bufB + 1) & ~1);   // the template's band sums of this chunk, all bands (16-byte aligned)
  const int B = p.B, ob = p.out_band;

  // stage every band's sums at once (one round of HBM latency for the whole template): a template with one
  // unit in a band gets that row as ONE TMA bulk copy (thread 0 issues them, completion on an mbarrier: the
  // LSU path of per-thread cp.async tops out near 14 GB/s per SM here), more units are added up on the way
  __shared__ uint64_t cbar;
  // the interpolator histories of every band, requested up front: read stage by stage they were six serialised
  // global-memory latencies on the critical path of a CTA (long_scoreboard 3.9 per issue, profiles/r2 section 4)
  __shared__ float2 hsm[SPIIR_MAX_BANDS][kUpHist + 1];
  for (int i = tid; i < SPIIR_MAX_BANDS * kUpHist; i += kCombineThreads) {
    const int b = i / kUpHist, j = i - b * kUpHist;
    if (b > ob && b < B) hsm[b][j] = p.uphist[b][((size_t)det * p.T + t) * kUpHist + j];
  }
  if (tid == 0) mbar_init(&cbar, 1);
  __syncthreads();
  if (tid == 0) {
    uint32_t bytes = 0;
    for (int b = 0; b < B; ++b)
      if (p.tb_count[t * B + b] == 1) bytes += (uint32_t)p.sb_n[b] * 8u;
    mbar_expect_tx(&cbar, bytes);
    for (int b = 0; b < B; ++b)
      if (p.tb_count[t * B + b] == 1)
        tma_load_1d(sbuf + p.sb_off[b],
                    p.S[b] + (size_t)det * p.S_det_stride[b] + (size_t)p.tb_first[t * B + b] * p.nmax[b],
                    (uint32_t)p.sb_n[b] * 8u, &cbar);
  }
  for (int b = 0; b < B; ++b) {
    const int ns = p.sb_n[b];                           // samples k_bank stored for this band (n, or n/2 if odd-only)
    const float2* S = p.S[b] + (size_t)det * p.S_det_stride[b];
    const int first = p.tb_first[t * B + b], count = p.tb_count[t * B + b];
    float2* dst = sbuf + p.sb_off[b];
    if (count != 1)
      for (int m = tid; m < ns; m += kCombineThreads) dst[m] = unit_sum(S, p.nmax[b], first, count, m);
  }
  mbar_wait(&cbar, 0);
  __syncthreads();

  // acc_{B-1} = s_{B-1}, then acc_b = s_b + up2(acc_{b+1}) down to the output band
  for (int b = B - 1; b >= ob; --b) {
    float2* cur = buf[(b - ob) & 1];
    const int n = p.n[b];
    const float2* sb = sbuf + p.sb_off[b];
    float2* hist = (b > ob) ? p.uphist[b] + ((size_t)det * p.T + t) * kUpHist : nullptr;
    if (hist && tid < kUpHist) cur[tid] = hsm[b][tid];
    if (b == B - 1) {
      for (int m = tid; m < n; m += kCombineThreads) cur[kUpHist + m] = sb[m];
    } else {
      // four outputs per thread from one 17-sample window of acc_{b+1} held in registers:
      // m = 2j, 2j+1 share the window ending at acc[j], m = 2j+2, 2j+3 the one ending at acc[j+1]
      const float2* src = buf[(b + 1 - ob) & 1];
      for (int j0 = 2 * tid; 2 * j0 < n; j0 += 2 * kCombineThreads) {
        float2 w[18];
#pragma unroll
        for (int i = 0; i < 9; ++i) {
          const float4 v = *reinterpret_cast<const float4*>(src + j0 + 2 * i);     // src[j0 + i] = acc[j0 + i - 15]
          w[2 * i] = make_float2(v.x, v.y); w[2 * i + 1] = make_float2(v.z, v.w);
        }
        const float4 s01 = *reinterpret_cast<const float4*>(sb + 2 * j0);
        const float4 s23 = *reinterpret_cast<const float4*>(sb + 2 * j0 + 2);
        float2 a0 = make_float2(s01.x, s01.y), a1 = make_float2(s01.z, s01.w);
        float2 a2 = make_float2(s23.x, s23.y), a3 = make_float2(s23.z, s23.w);
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const float2 he = make_float2(hr[2 * q], hr[2 * q]), ho = make_float2(hr[2 * q + 1], hr[2 * q + 1]);
          const float2 u = w[15 - q], v = w[16 - q];
          a0 = __ffma2_rn(he, u, a0);                       // packed (re, im): half the issue slots
          a1 = __ffma2_rn(ho, u, a1);
          a2 = __ffma2_rn(he, v, a2);
          a3 = __ffma2_rn(ho, v, a3);
        }
        float2* o = cur + kUpHist + 2 * j0;
        o[0] = a0; o[1] = a1; o[2] = a2; o[3] = a3;
      }
    }
    __syncthreads();
    if (hist && tid < kUpHist) hist[tid] = cur[n + tid];       // last 15 of [old history | new samples]
  }

  // output samples, ring append, fused per-template maximum (H4 mode 0)
  const float2* acc = buf[0] + kUpHist;
  const int n_out = p.n_out;
  const float2* s0 = sbuf + p.sb_off[0];                        // ob == 1: s_0[2m+1] stored at index m
  float2* ring = p.ring + (size_t)det * p.ring_det_stride + (size_t)t * p.ring_len;
  float2* out = p.snr_out ? p.snr_out + ((size_t)det * p.T + t) * n_out : nullptr;
  float best = -1.f; int bk = 0; float2 bz = make_float2(0.f, 0.f);
  const long long kbase = p.k0 % p.ring_len;           // n_out <= ring_len: one conditional wrap per sample
  for (int m = tid; m < n_out; m += kCombineThreads) {
    float2 z = acc[m];
    if (ob == 1) {                                             // band 0 runs at twice the output rate (M5)
      const float2 v = s0[m];
      z.x += v.x; z.y += v.y;
    }
    long long kk = kbase + m;
    if (kk >= p.ring_len) kk -= p.ring_len;
    ring[kk] = z;
    if (out) out[m] = z;
    const float m2 = __fadd_rn(__fmul_rn(z.x, z.x), __fmul_rn(z.y, z.y));
    if (m2 > best) { best = m2; bk = m; bz = z; }
  }
  const int mybk = bk;
  // block arg-max, lowest k on ties
  for (int o = 16; o; o >>= 1) {
    const float om = __shfl_xor_sync(0xffffffffu, best, o);
    const int ok = __shfl_xor_sync(0xffffffffu, bk, o);
    if (om > best || (om == best && ok < bk)) { best = om; bk = ok; }
  }
  if ((tid & 31) == 0) { red_m2[tid >> 5] = best; red_k[tid >> 5] = bk; }
  __syncthreads();
  float fb = red_m2[0]; int fk = red_k[0];
  for (int wv = 1; wv < kCombineThreads / 32; ++wv)
    if (red_m2[wv] > fb || (red_m2[wv] == fb && red_k[wv] < fk)) { fb = red_m2[wv]; fk = red_k[wv]; }
  if (fk % kCombineThreads == tid && fb >= 0.f) {              // the thread that owns sample fk holds its z
    // bz belongs to this thread's own best; recompute from the ring if they differ
    float2 z = (mybk == fk) ? bz : ring[(p.k0 + fk) % p.ring_len];
    PeakRec rec; rec.k = p.k0 + fk; rec.zr = z.x; rec.zi = z.y; rec.m2 = fb; rec._pad = 0;
    p.peak[(size_t)det * p.T + t] = rec;
  }
}

int launch_combine(const CombineParams& p, int n_det, cudaStream_t st) {
  static unsigned long long configured = 0;
  if (first_use_on_device(configured)) {
    SPIIR_CUDA_OK(cudaFuncSetAttribute(k_combine, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  }
  const size_t smem = (size_t)(((p.bufA + p.bufB + 1) & ~1) + p.sb_total) * sizeof(float2);
  k_combine<<<dim3(p.T, n_det), kCombineThreads, smem, st>>>(p);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

}  // namespace spiir
