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
//     direction of one tuple gathers the SAME samples.  The plan sorts the directions
//     of each trigger detector T by delay tuple into a stream of 32-slot chunks, one
//     slot per direction: the projector M = U2 U2^T in the order the kernel consumes
//     it, the pixel, and a control word (shared-memory rows to gather + which
//     detectors' rows changed since the previous slot).  On a change a thread
//     refreshes the real products q_IJ = Re(z_I conj z_J) the changed rows enter; each
//     direction then costs one N_q-term dot product (1 FMUL + 5 FFMA for three
//     detectors, issued for two pairs at a time as packed FFMA2 with the weight as a
//     scalar-broadcast operand) and one FMNMX3 per TWO directions for the running
//     maximum.  Which direction holds the maximum is recovered afterwards by rescanning
//     the one chunk that last raised it.
//   * thread = K (trigger, slide) pairs; a CTA owns 32 K pairs whose delay windows
//     (the only samples any direction can touch) sit in shared memory, pair-major:
//     one TMA bulk copy per (pair, detector) window (cp.async.bulk + mbarrier; 8-byte
//     cp.async when the view is not 16-byte friendly); each warp takes a contiguous
//     share of the stream's chunks and stages each chunk through shared memory for
//     broadcast reads.
//   * valid trigger slots are binned by trigger detector on the device (no host sync);
//     one launch per trigger detector, persistent CTAs stride over the pair batches.
#include <algorithm>
#include <climits>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "sky_internal.cuh"

namespace spiir {

constexpr int kSkyKMax = 4;                 // (trigger, slide) pairs per thread, at most

template <int D> struct SkyFmt {
  static constexpr int NO = D - 1;                       // detectors other than the trigger detector
  static constexpr int NQ = D * (D + 1) / 2;             // independent entries of the projector
  static constexpr int SW = (NQ + 1 + 3) / 4 * 4;        // words per slot: NQ - 1 weights + control + pixel, padded to 16 B
};
// One slot per direction, SW words: words [0, NQ-1) weights, word NQ-1 = control, word NQ = pixel.
//   The weight of |z_T|^2 is not stored: the projector has trace 2, so M_TT = 2 - sum_o M_oo and the kernel evaluates
//   rho_c^2 - 2 |z_T|^2 = sum_o M_oo (|z_o|^2 - |z_T|^2) + cross terms.  Weight order (T = trigger detector, o = others
//   in increasing detector index): M_oo (o = 0..NO-1); 2 M_To; 2 M_o'o for o' < o, (0,1) (0,2) (1,2).
//   Weights and control come first so that the main loop reads NQ words per slot — for three detectors one LDS.128 and
//   one LDS.64 (3 shared-memory wavefronts per warp instead of 4: the broadcast reads of the slot are half of the
//   kernel's shared-memory traffic, which co-limits it with the FP32 pipe; profiles/r2_ncu_summary.md section 2).
//   control = nref | f_0 << 2 | f_1 << 12 | f_2 << 22: f_o = element offset, inside a pair's block of
//   windows, of the sample of other detector o this direction reads (segment offset + row, < 1024);
//   nref = NO - (first other detector whose row differs from the previous slot): the last nref
//   detectors are refreshed (NO for the first slot of a warp's share of the stream: refresh
//   everything; 0: same delay tuple, nothing to refresh — one bit test on the common path).
// The last chunk is padded with copies of the last direction (nref 0).

struct SkyParams {
  const float* stream; int32_t n_chunks;                      // this trigger detector's stream
  int32_t cb[kSkyWarps + 1];                                  // chunks [cb[w], cb[w+1]) are warp w's share (balanced by cost)
  int32_t n_pix;
  const float2* z; int64_t det_stride, row_stride, ring_len, k_newest;
  const spiir_trigger* trig;
  const SkyRec* list; const int32_t* counts;                  // candidates of trigger detector T
  int32_t T;
  int32_t n_slides;                                           // 0 = foreground
  int64_t step; int32_t mult[SPIIR_MAX_DET];
  int32_t lo[SPIIR_MAX_DET], W[SPIIR_MAX_DET], woff[SPIIR_MAX_DET];   // window of detector I vs T: first delta, width, first row
  int32_t win_elems;                                          // float2 elements of the window region
  int32_t ps;                                                 // float2 elements of one pair's block of windows (even)
  int32_t soff[SPIIR_MAX_DET];                                // offset of detector I's segment in the block (even)
  int32_t tma;                                                // view is 16-byte friendly: stage with TMA bulk copies
  spiir_sky_result* out; float* map;
};

struct PairInfo { int32_t slot, slide, valid, row; float2 vT; long long k; unsigned char sh[8]; };   // sh[I]: 0/1 sample shift of detector I's window (TMA copies start 16-byte aligned)

template <int NQ>
__device__ __forceinline__ float quad_form(const float* __restrict__ w, const float (&q)[NQ]) {
  float c = __fmul_rn(w[0], q[1]);                     // the term of q[0] = |z_T|^2 is the constant 2 q[0] (trace of the projector)
#pragma unroll
  for (int e = 2; e < NQ; ++e) c = __fmaf_rn(w[e - 1], q[e], c);
  return c;
}

template <int D, int K, bool MAP>
__global__ void __launch_bounds__(kSkyThreads, 1) k_sky(const __grid_constant__ SkyParams P) {
  constexpr int NO = SkyFmt<D>::NO, NQ = SkyFmt<D>::NQ, SW = SkyFmt<D>::SW;
  constexpr int NP = 32 * K;
  const int PS = P.ps;                                 // float2 elements of a pair's block of windows
  constexpr int kTileWords = (kSkyChunk * SW > 2 * NP) ? kSkyChunk * SW : 2 * NP;   // a warp's chunk tile, reused for the reduction
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* win = reinterpret_cast<float2*>(smem_raw);                              // [pair][PS]: a pair's windows, detector after detector
  float* tiles = reinterpret_cast<float*>(win + P.win_elems);                     // [warps][kTileWords]
  PairInfo* pinfo = reinterpret_cast<PairInfo*>(tiles + kSkyWarps * kTileWords);  // [NP]
  int* wchunk = reinterpret_cast<int*>(pinfo + NP);                               // [NP] chunk holding each pair's maximum

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int T = P.T;
  const int S1 = P.n_slides > 0 ? P.n_slides : 1;
  const long long n_pairs = (long long)P.counts[T] * S1;
  const long long n_batches = (n_pairs + NP - 1) / NP;
  const int64_t kmin = (P.k_newest - P.ring_len + 1 > 0) ? P.k_newest - P.ring_len + 1 : 0;
  float* mytile = tiles + warp * kTileWords;
  // a contiguous share of chunks per warp: only a share's first slot has to refresh everything
  const int c_beg = P.cb[warp], c_end = P.cb[warp + 1];

  __shared__ uint64_t bar;                             // completion of a batch's TMA window copies
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(&bar)), "r"(NP * NO));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  uint32_t bar_phase = 0;

  for (long long batch = blockIdx.x; batch < n_batches; batch += gridDim.x) {
    __syncthreads();                                   // previous batch fully consumed
    // ---- pair set-up: which trigger, which slide, is every gather inside the view
    if (tid < NP) {
      PairInfo pi; pi.slot = -1; pi.slide = 0; pi.valid = 0; pi.row = 0; pi.vT = make_float2(0.f, 0.f); pi.k = 0;
      const long long q = batch * NP + tid;
      if (q < n_pairs) {
        const SkyRec rc = P.list[q / S1];
        pi.slot = rc.slot;
        pi.slide = (int)(q % S1) + (P.n_slides > 0 ? 1 : 0);
        pi.row = rc.row; pi.k = rc.k;
        bool ok = rc.k_ok != 0;
#pragma unroll
        for (int I = 0; I < D; ++I) {
          if (I == T) continue;
          const int64_t k0 = rc.k - (int64_t)pi.slide * P.step * P.mult[I] + P.lo[I];
          ok = ok && k0 >= kmin && k0 + P.W[I] - 1 <= P.k_newest;
        }
        pi.valid = ok ? 1 : 0;
        if (ok) pi.vT = rc.vT;
      }
      pinfo[tid] = pi;
    }
    __syncthreads();
    // the warp's first chunk of the direction stream does not depend on the batch: request it now, it arrives
    // while the windows are staged
    float4 pre[SW / 4];
    if (c_beg < c_end) {
      const float4* src = reinterpret_cast<const float4*>(P.stream + ((size_t)c_beg * kSkyChunk + lane) * SW);
#pragma unroll
      for (int c = 0; c < SW / 4; ++c) pre[c] = __ldg(src + c);
    }
    // ---- delay windows -> shared memory, pair-major.  With a 16-byte friendly view one thread per (pair,
    //      detector) issues the window as one TMA bulk copy (two if it wraps the ring), starting at the
    //      16-byte aligned sample at or before the window (sh = 0/1 samples of shift); completion on an
    //      mbarrier.  Otherwise warps copy the windows with 8-byte cp.async.
    if (P.tma) {
      // the windows were last written through the generic proxy (zero fill, in-place shift); the bulk copies below
      // write them through the async proxy
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      if (tid < NP * NO) {
        const int j = tid / NO, o = tid - j * NO;
        const int I = o + (o >= T ? 1 : 0);
        const PairInfo pi = pinfo[j];
        const uint32_t bar_a = (uint32_t)__cvta_generic_to_shared(&bar);
        float2* dst = win + (size_t)j * PS + P.soff[I];
        if (pi.valid) {
          const int64_t k0 = pi.k - (int64_t)pi.slide * P.step * P.mult[I] + P.lo[I];
          const int64_t base = k0 % P.ring_len;
          const int sh = (int)(base & 1);
          const int64_t idx0 = base - sh;
          const int len = (P.W[I] + sh + 1) & ~1;                    // samples copied: even, covers the window
          const int n1 = (int)min((int64_t)len, P.ring_len - idx0);  // before the ring's end (even: ring_len is even)
          const float2* row = P.z + (size_t)I * P.det_stride + (size_t)pi.row * P.row_stride;
          pinfo[j].sh[I] = (unsigned char)sh;
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(len * 8) : "memory");
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                           (uint32_t)__cvta_generic_to_shared(dst)), "l"(row + idx0), "r"(n1 * 8), "r"(bar_a) : "memory");
          if (n1 < len)
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                             (uint32_t)__cvta_generic_to_shared(dst + n1)), "l"(row), "r"((len - n1) * 8), "r"(bar_a) : "memory");
        } else {
          for (int r = 0; r < P.W[I] + 2; ++r) dst[r] = make_float2(0.f, 0.f);
          pinfo[j].sh[I] = 0;
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar_a) : "memory");
        }
      }
      mbar_wait_bounded((uint32_t)__cvta_generic_to_shared(&bar), bar_phase);
      bar_phase ^= 1u;
      // the copies landed with sample k0 at offset sh (0/1, from the source's alignment); move each window
      // so that it starts at the parity its lane wants: lanes l and l+8 of a half-warp then hit distinct banks
      for (int task = warp; task < NP * NO; task += kSkyWarps) {
        const int j = task / NO, o = task - j * NO;
        const int I = o + (o >= T ? 1 : 0);
        const int sh = pinfo[j].sh[I], par = (j >> 3) & 1;
        if (sh != par) {
          float2* seg = win + (size_t)j * PS + P.soff[I];
          const int W = P.W[I], nblk = (W + 127) >> 7;
          for (int bq = 0; bq < nblk; ++bq) {              // 128 samples at a time, in the direction that never
            const int r0 = ((par < sh) ? bq : nblk - 1 - bq) << 7;   // overwrites a sample still to be moved
            float2 t[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { const int r = r0 + lane + 32 * u; if (r < W) t[u] = seg[sh + r]; }
            __syncwarp();
#pragma unroll
            for (int u = 0; u < 4; ++u) { const int r = r0 + lane + 32 * u; if (r < W) seg[par + r] = t[u]; }
            __syncwarp();
          }
        }
      }
    } else {
      for (int task = warp; task < NP * NO; task += kSkyWarps) {
        const int j = task / NO, o = task - j * NO;
        const int I = o + (o >= T ? 1 : 0);
        const PairInfo pi = pinfo[j];
        const int W = P.W[I];
        float2* dst = win + (size_t)j * PS + P.soff[I] + ((j >> 3) & 1);
        if (pi.valid) {
          const int64_t k0 = pi.k - (int64_t)pi.slide * P.step * P.mult[I] + P.lo[I];
          const int64_t base = k0 % P.ring_len;
          const float2* src = P.z + (size_t)I * P.det_stride + (size_t)pi.row * P.row_stride;
          for (int r = lane; r < W; r += 32) {
            int64_t idx = base + r;
            if (idx >= P.ring_len) idx -= P.ring_len;
            cp_async_8(dst + r, src + idx);
          }
        } else {
          for (int r = lane; r < W; r += 32) dst[r] = make_float2(0.f, 0.f);
        }
      }
      cp_async_wait_all();
    }
    __syncthreads();

    // ---- the direction stream: this warp's chunks.  Only the running maximum is kept per direction
    //      (one FMNMX3 per two directions); which chunk raised it last is noted per chunk, and that chunk is rescanned below.
    float2 vT[K], v[NO][K];
    float best[K], seen[K]; int bch[K];
    float2 qp[(K + 1) / 2][NQ];                          // products of pairs (2i, 2i+1) side by side: packed FFMA2 operands
#define SKY_Q(a, e) (((a) & 1) ? qp[(a) >> 1][e].y : qp[(a) >> 1][e].x)
    long long mrow[K];                                  // sky-map row of each pair, -1 = none
    uint32_t pb[K];                                     // shared-space byte address of pair a's block, plus its windows' parity
#pragma unroll
    for (int a = 0; a < K; ++a) {
      const PairInfo pi = pinfo[lane + 32 * a];
      pb[a] = (uint32_t)__cvta_generic_to_shared(win + (lane + 32 * a) * PS + ((lane >> 3) & 1));
      vT[a] = pi.vT; best[a] = -3.0e38f; seen[a] = -3.0e38f; bch[a] = c_beg;
      mrow[a] = (MAP && pi.valid) ? (long long)pi.slot * P.n_pix : -1;
#pragma unroll
      for (int e = 0; e < NQ; ++e) SKY_Q(a, e) = 0.f;
      SKY_Q(a, 0) = re_prod(vT[a], vT[a]);
#pragma unroll
      for (int o = 0; o < NO; ++o) v[o][a] = make_float2(0.f, 0.f);
    }

    for (int ch = c_beg; ch < c_end; ++ch) {
      __syncwarp();
#pragma unroll
      for (int c = 0; c < SW / 4; ++c) reinterpret_cast<float4*>(mytile + lane * SW)[c] = pre[c];
      __syncwarp();
      if (ch + 1 < c_end) {                                   // prefetch the next chunk while this one is consumed
        const float4* src = reinterpret_cast<const float4*>(P.stream + ((size_t)(ch + 1) * kSkyChunk + lane) * SW);
#pragma unroll
        for (int c = 0; c < SW / 4; ++c) pre[c] = __ldg(src + c);
      }
      // words of a slot the loop needs: NQ - 1 weights and the control word (and the pixel for the sky map), read as
      // N4 float4 and, when two words or fewer remain, one float2
      constexpr int LW = NQ + (MAP ? 1 : 0);
      constexpr bool H2 = (LW % 4 == 1 || LW % 4 == 2);
      constexpr int N4 = H2 ? LW / 4 : (LW + 3) / 4;
      float4 nxt[N4 > 0 ? N4 : 1]; float2 nxt2 = make_float2(0.f, 0.f);
#pragma unroll
      for (int c = 0; c < N4; ++c) nxt[c] = reinterpret_cast<const float4*>(mytile)[c];
      if (H2) nxt2 = reinterpret_cast<const float2*>(mytile)[2 * N4];
      float pend[K];
#pragma unroll 4
      for (int s = 0; s < kSkyChunk; ++s) {
        float w[SW + 2];
#pragma unroll
        for (int c = 0; c < N4; ++c) { w[4 * c] = nxt[c].x; w[4 * c + 1] = nxt[c].y; w[4 * c + 2] = nxt[c].z; w[4 * c + 3] = nxt[c].w; }
        if (H2) { w[4 * N4] = nxt2.x; w[4 * N4 + 1] = nxt2.y; }
        // the next slot is fetched (broadcast read) before this one is consumed
        const float* nslot = mytile + ((s + 1) & (kSkyChunk - 1)) * SW;
#pragma unroll
        for (int c = 0; c < N4; ++c) nxt[c] = reinterpret_cast<const float4*>(nslot)[c];
        if (H2) nxt2 = reinterpret_cast<const float2*>(nslot)[2 * N4];
        const int ctrl = __float_as_int(w[NQ - 1]);
        const int nref = ctrl & 3;
        if (nref) {
          // new delay tuple: gather the rows that changed, refresh the products they enter
#pragma unroll
          for (int o = 0; o < NO; ++o) {
            if (o >= NO - nref) {
              // 32-bit shared-space addresses: one IADD per gather instead of a 64-bit generic address
              const uint32_t ro = (uint32_t)((ctrl >> (2 + kSkyRowBits * o)) & ((1 << kSkyRowBits) - 1)) * 8u;
#pragma unroll
              for (int a = 0; a < K; ++a) {
                const float2 x = lds64(pb[a] + ro);
                v[o][a] = x;
                SKY_Q(a, 1 + o) = __fsub_rn(re_prod(x, x), SKY_Q(a, 0));
                SKY_Q(a, 1 + NO + o) = re_prod(vT[a], x);
#pragma unroll
                for (int o2 = 0; o2 < o; ++o2) SKY_Q(a, 1 + 2 * NO + o * (o - 1) / 2 + o2) = re_prod(v[o2][a], x);
              }
            }
          }
        }
        // the quadratic form of two pairs at a time: scalar weight x packed products (FFMA2, the same
        // per-component roundings as quad_form in the rescan)
        float cval[K];
#pragma unroll
        for (int i = 0; i < K / 2; ++i) {
          float2 c2 = __fmul2_rn(make_float2(w[0], w[0]), qp[i][1]);
#pragma unroll
          for (int e = 2; e < NQ; ++e) c2 = __ffma2_rn(make_float2(w[e - 1], w[e - 1]), qp[i][e], c2);
          cval[2 * i] = c2.x; cval[2 * i + 1] = c2.y;
        }
        if (K & 1) {
          float c = __fmul_rn(w[0], qp[K / 2][1].x);
#pragma unroll
          for (int e = 2; e < NQ; ++e) c = __fmaf_rn(w[e - 1], qp[K / 2][e].x, c);
          cval[K - 1] = c;
        }
#pragma unroll
        for (int a = 0; a < K; ++a) {
          if (MAP) {
            if (mrow[a] >= 0) P.map[mrow[a] + __float_as_int(w[NQ])] = __fmaf_rn(2.f, SKY_Q(a, 0), cval[a]);
          }
          // two directions per maximum: the value of an even slot waits for its odd neighbour (one FMNMX3)
          if (s & 1) best[a] = fmax3(best[a], pend[a], cval[a]);
          else       pend[a] = cval[a];
        }
      }
#undef SKY_Q
#pragma unroll
      for (int a = 0; a < K; ++a)
        if (best[a] > seen[a]) { seen[a] = best[a]; bch[a] = ch; }
    }
    __syncthreads();                                   // every warp is done with its tile: reuse it for the reduction
    {
      float* red_c = mytile; int* red_i = reinterpret_cast<int*>(mytile + NP);
#pragma unroll
      for (int a = 0; a < K; ++a) { red_c[lane + 32 * a] = best[a]; red_i[lane + 32 * a] = bch[a]; }
    }
    __syncthreads();
    // ---- across the warps: thread = pair, the first warp (= earliest chunks of the stream) wins exact ties
    if (tid < NP) {
      float bc = tiles[tid]; int bi = reinterpret_cast<const int*>(tiles + NP)[tid];
#pragma unroll 4
      for (int wv = 1; wv < kSkyWarps; ++wv) {
        const float c = tiles[wv * kTileWords + tid];
        const int i = reinterpret_cast<const int*>(tiles + wv * kTileWords + NP)[tid];
        if (c > bc) { bc = c; bi = i; }
      }
      wchunk[tid] = min(bi, P.n_chunks - 1);
    }
    __syncthreads();
    // ---- then a warp rescans the winning chunk of each of its 2 K pairs, lane = slot (the chunks of four
    //      pairs are requested before the first is consumed): every lane forms its own direction's products
    //      from scratch, the first lane holding the maximum gives the direction, tot2 and null2 there (Eq. 10)
    //      The pairs of a warp are taken RB at a time in three passes — every pair's value first, then the five
    //      shuffle steps of all RB maxima side by side, then the results — so that the shuffle latencies overlap.
    constexpr int PPW = NP / kSkyWarps;
    constexpr int RB = (PPW * (SW / 4) <= 16) ? PPW : ((PPW % 4 == 0) ? 4 : 2);
    for (int u0 = 0; u0 < PPW; u0 += RB) {
      float4 wv4[RB][SW / 4];
#pragma unroll
      for (int u = 0; u < RB; ++u) {
        const float4* sp = reinterpret_cast<const float4*>(
            P.stream + ((size_t)wchunk[warp + (u0 + u) * kSkyWarps] * kSkyChunk + lane) * SW);
#pragma unroll
        for (int c = 0; c < SW / 4; ++c) wv4[u][c] = __ldg(sp + c);
      }
      float cc[RB], cm[RB], tt[RB], q0[RB]; int px[RB], slot[RB], slide[RB], valid[RB];
#pragma unroll
      for (int u = 0; u < RB; ++u) {
        const int j = warp + (u0 + u) * kSkyWarps;
        const PairInfo pi = pinfo[j];
        slot[u] = pi.slot; slide[u] = pi.slide; valid[u] = pi.valid;
        float w[SW];
#pragma unroll
        for (int c = 0; c < SW / 4; ++c) {
          w[4 * c] = wv4[u][c].x; w[4 * c + 1] = wv4[u][c].y; w[4 * c + 2] = wv4[u][c].z; w[4 * c + 3] = wv4[u][c].w;
        }
        const int ctrl = __float_as_int(w[NQ - 1]);
        float qq[NQ]; float2 vv[NO];
        qq[0] = re_prod(pi.vT, pi.vT);
        float tot = qq[0];
#pragma unroll
        for (int o = 0; o < NO; ++o) {
          const float2 x = win[(size_t)j * PS + ((j >> 3) & 1) +
                               ((ctrl >> (2 + kSkyRowBits * o)) & ((1 << kSkyRowBits) - 1))];
          vv[o] = x;
          const float xx = re_prod(x, x);
          qq[1 + o] = __fsub_rn(xx, qq[0]);
          qq[1 + NO + o] = re_prod(pi.vT, x);
#pragma unroll
          for (int o2 = 0; o2 < o; ++o2) qq[1 + 2 * NO + o * (o - 1) / 2 + o2] = re_prod(vv[o2], x);
          tot += xx;
        }
        cc[u] = quad_form<NQ>(w, qq); cm[u] = cc[u]; tt[u] = tot; q0[u] = qq[0]; px[u] = __float_as_int(w[NQ]);
      }
#pragma unroll
      for (int o = 16; o; o >>= 1) {
#pragma unroll
        for (int u = 0; u < RB; ++u) cm[u] = fmaxf(cm[u], __shfl_xor_sync(0xffffffffu, cm[u], o));
      }
#pragma unroll
      for (int u = 0; u < RB; ++u) {
        const int src = __ffs(__ballot_sync(0xffffffffu, cc[u] == cm[u])) - 1;
        const float tot2 = __shfl_sync(0xffffffffu, tt[u], src);
        const int pix = __shfl_sync(0xffffffffu, px[u], src);
        if (slot[u] < 0) continue;
        spiir_sky_result res; res.coh2 = 0.f; res.null2 = 0.f; res.tot2 = 0.f; res.pix = -1;
        if (valid[u]) {
          res.coh2 = __fmaf_rn(2.f, q0[u], cm[u]);
          res.tot2 = tot2;
          res.pix = pix;
          res.null2 = fmaxf(res.tot2 - res.coh2, 0.f);
        }
        if (lane == 0) P.out[(size_t)slot[u] * S1 + (P.n_slides > 0 ? slide[u] - 1 : 0)] = res;
      }
    }
  }
}

// valid slots -> per-detector lists; invalid slots get their "no result" rows here
__global__ void __launch_bounds__(256) k_sky_bin(const spiir_trigger* trig, int n_slots, int n_det, int S1,
                                                 const float2* z, int64_t det_stride, int64_t row_stride,
                                                 int64_t ring_len, int64_t k_newest, int64_t n_rows,
                                                 SkyRec* lists, int32_t* counts, int max_slots,
                                                 spiir_sky_result* out) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  if (i >= n_slots) return;
  const spiir_trigger t = trig[i];
  if (t.valid && t.det >= 0 && t.det < n_det && t.tmpl >= 0 && t.tmpl < n_rows) {   // a stale or garbage slot never indexes the view
    const int64_t kmin = (k_newest - ring_len + 1 > 0) ? k_newest - ring_len + 1 : 0;
    SkyRec rc;
    rc.slot = i; rc.row = t.tmpl; rc.k = t.k; rc._pad = 0;
    rc.k_ok = (t.k >= kmin && t.k <= k_newest) ? 1 : 0;
    rc.vT = rc.k_ok ? z[(size_t)t.det * det_stride + (size_t)t.tmpl * row_stride + (size_t)(t.k % ring_len)]
                    : make_float2(0.f, 0.f);
    const int pos = atomicAdd(counts + t.det, 1);
    lists[(size_t)t.det * max_slots + pos] = rc;
  } else {
    spiir_sky_result r; r.coh2 = 0.f; r.null2 = 0.f; r.tot2 = 0.f; r.pix = -1;
    for (int s = 0; s < S1; ++s) out[(size_t)i * S1 + s] = r;
  }
}

}  // namespace spiir

using namespace spiir;

static size_t sky_align(size_t x) { return (x + 255) / 256 * 256; }
static int sky_slot_words(int D) { return (D * (D + 1) / 2 + 1 + 3) / 4 * 4; }
static int sky_win_elems(int ps, int K) { return ps * 32 * K; }          // ps is even
static size_t sky_smem_bytes(int ps, int SW, int K) {
  const int NP = 32 * K, tile = std::max(kSkyChunk * SW, 2 * NP);
  return (size_t)sky_win_elems(ps, K) * 8 + (size_t)kSkyWarps * tile * 4 + (size_t)NP * (sizeof(PairInfo) + 4);
}

static void sky_layout(spiir_sky_plan* pl) {
  const int D = pl->n_det;
  pl->SW = sky_slot_words(D);
  pl->cap_slots = (pl->n_pix + kSkyChunk - 1) / kSkyChunk * kSkyChunk;       // one slot per direction, whole chunks
  size_t cur = 0;
  for (int T = 0; T < D; ++T) {
    pl->st[T].off_slots = cur; cur = sky_align(cur + (size_t)pl->cap_slots * pl->SW * 4);
  }
  pl->off_lists = cur;  cur = sky_align(cur + (size_t)D * pl->max_slots * sizeof(SkyRec));
  pl->off_counts = cur; cur = sky_align(cur + SPIIR_MAX_DET * 4);
  pl->bytes = cur;
}

// Builds the chunked stream of trigger detector T on the host.
static void sky_build_stream(spiir_sky_plan* pl, int T, const float* u2, const int32_t* delay,
                             std::vector<float>& slots) {
  const int D = pl->n_det, NO = D - 1, NQ = D * (D + 1) / 2, SW = pl->SW, n_pix = pl->n_pix;
  spiir_sky_stream& S = pl->st[T];
  int oth[SPIIR_MAX_DET];
  for (int o = 0; o < NO; ++o) oth[o] = o + (o >= T ? 1 : 0);
  std::vector<int32_t> rows((size_t)n_pix * 3, 0);
  for (int p = 0; p < n_pix; ++p)
    for (int o = 0; o < NO; ++o) {
      const int I = oth[o];
      rows[(size_t)p * 3 + o] = S.woff[I] + (delay[(size_t)p * D + I] - delay[(size_t)p * D + T] - S.lo[I]);
    }
  // directions sorted by delay tuple, then by pixel index
  std::vector<int32_t> order(n_pix);
  for (int p = 0; p < n_pix; ++p) order[p] = p;
  std::sort(order.begin(), order.end(), [&](int32_t x, int32_t y) {
    for (int o = 0; o < 3; ++o)
      if (rows[(size_t)x * 3 + o] != rows[(size_t)y * 3 + o]) return rows[(size_t)x * 3 + o] < rows[(size_t)y * 3 + o];
    return x < y;
  });
  // how many of the other detectors' rows each slot refreshes (the last ones), before the warps' shares are cut
  const int n_chunks = pl->cap_slots / kSkyChunk;
  std::vector<int> nrf(pl->cap_slots, 0);
  S.n_tuples = 0;
  for (int r = 0; r < n_pix; ++r) {
    int level = 0;
    if (r > 0) {
      const int32_t* pr = &rows[(size_t)order[r - 1] * 3];
      const int32_t* rw = &rows[(size_t)order[r] * 3];
      while (level < NO && pr[level] == rw[level]) ++level;
    }
    nrf[r] = NO - level;
    if (nrf[r]) ++S.n_tuples;
  }
  // the 16 warps take contiguous runs of chunks of about equal COST (a refreshed row costs about as much as one
  // direction and a half): the warps whose share is dense in delay tuples no longer finish last
  {
    std::vector<double> cost(n_chunks, 0.0);
    double total = 0;
    for (int c = 0; c < n_chunks; ++c) {
      double x = kSkyChunk;
      for (int r = c * kSkyChunk; r < (c + 1) * kSkyChunk; ++r) x += 1.5 * nrf[r];
      cost[c] = x; total += x;
    }
    double acc = 0; int wv = 1;
    S.cb[0] = 0;
    for (int c = 0; c < n_chunks && wv < kSkyWarps; ++c) {
      acc += cost[c];
      if (acc >= total * wv / kSkyWarps) S.cb[wv++] = c + 1;
    }
    for (; wv <= kSkyWarps; ++wv) S.cb[wv] = n_chunks;
  }
  slots.assign((size_t)pl->cap_slots * SW, 0.f);
  for (int r = 0; r < pl->cap_slots; ++r) {
    float* w = &slots[(size_t)r * SW];
    if (r >= n_pix) {                      // padding: the last direction again, nothing to refresh
      memcpy(w, w - SW, (size_t)SW * 4);
      int32_t ctrl; memcpy(&ctrl, w + NQ - 1, 4);
      ctrl &= ~3;
      memcpy(w + NQ - 1, &ctrl, 4);
      continue;
    }
    const int p = order[r];
    const int32_t* rw = &rows[(size_t)p * 3];
    int nref = nrf[r];
    for (int wv = 0; wv < kSkyWarps; ++wv)
      if (r == S.cb[wv] * kSkyChunk) nref = NO;   // a warp's share of the stream starts from nothing
    const float* u = u2 + (size_t)p * D * 2;
    auto M = [&](int I, int J) { return (double)u[2 * I] * u[2 * J] + (double)u[2 * I + 1] * u[2 * J + 1]; };
    // projector U2 U2^T in float64 from the float32 table, rounded once, in the kernel's order.
    // U2 has orthonormal columns (Eq. 27: the left singular vectors), so the projector has trace 2 and
    // M_TT = 2 - sum_o M_oo: the kernel evaluates rho_c^2 - 2 |z_T|^2 = sum_o M_oo (|z_o|^2 - |z_T|^2) + cross terms,
    // one multiply-add fewer per direction, and adds the constant back at the end
    {
      double tr = M(T, T);
      for (int o = 0; o < NO; ++o) tr += M(oth[o], oth[o]);
      if (!(tr > 2.0 - 1e-4 && tr < 2.0 + 1e-4)) S.bad_trace = 1;
    }
    for (int o = 0; o < NO; ++o) w[o] = (float)M(oth[o], oth[o]);
    for (int o = 0; o < NO; ++o) w[NO + o] = (float)(2.0 * M(T, oth[o]));
    for (int o = 1; o < NO; ++o)
      for (int o2 = 0; o2 < o; ++o2) w[2 * NO + o * (o - 1) / 2 + o2] = (float)(2.0 * M(oth[o2], oth[o]));
    int32_t ctrl = nref;                   // how many of the other detectors' rows to refresh, the last ones
    for (int o = 0; o < NO; ++o) ctrl |= rw[o] << (2 + kSkyRowBits * o);
    memcpy(w + NQ - 1, &ctrl, 4);
    const int32_t pix = p;
    memcpy(w + NQ, &pix, 4);
  }
  S.n_chunks = pl->cap_slots / kSkyChunk;
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
  const int D = n_det;
  pl->ws = (char*)dev_workspace;
  cudaStream_t st = (cudaStream_t)stream;
  std::vector<float> slots;
  for (int T = 0; T < D; ++T) {
    spiir_sky_stream& S = pl->st[T];
    int ps = 0;
    for (int I = 0; I < D; ++I) {
      int lo = INT_MAX, hi = INT_MIN;
      for (int p = 0; p < n_pix; ++p) {
        const long long d = (long long)delay[(size_t)p * D + I] - delay[(size_t)p * D + T];
        if (d < -1000000 || d > 1000000) { set_error("pixel %d: delay difference %lld out of range", p, d); delete pl; return SPIIR_EINVAL; }
        lo = std::min(lo, (int)d); hi = std::max(hi, (int)d);
      }
      // a detector's segment: its window, one sample of alignment shift, rounded up to an even length
      S.lo[I] = lo; S.W[I] = hi - lo + 1; S.woff[I] = ps;
      if (I != T) ps += (S.W[I] + 3) & ~1;
    }
    if (ps % 4 == 0) ps += 2;               // ps / 2 odd: a half-warp's 16 blocks start on distinct bank pairs
    S.rows = ps; S.ps = ps;
    S.k_max = 0;
    for (int K = kSkyKMax; K >= 1; --K)
      if (sky_smem_bytes(ps, pl->SW, K) <= (size_t)kSkySmemMax) { S.k_max = K; break; }
    if (S.k_max == 0) {
      set_error("delay span of trigger detector %d needs %zu bytes of shared memory (> %d)", T,
                sky_smem_bytes(ps, pl->SW, 1), kSkySmemMax);
      delete pl; return SPIIR_EINVAL;
    }
    if (ps >= (1 << kSkyRowBits)) {
      set_error("delay span of trigger detector %d: %d window samples do not fit the control word", T, ps);
      delete pl; return SPIIR_EINVAL;
    }
    S.bad_trace = 0;
    sky_build_stream(pl, T, u2, delay, slots);
    if (S.bad_trace) {
      set_error("host_u2: the two columns of U2 must be orthonormal at every pixel (Eq. 27: left singular vectors)");
      delete pl; return SPIIR_EINVAL;
    }
    cudaError_t e = cudaMemcpyAsync(pl->ws + S.off_slots, slots.data(), slots.size() * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);     // the host images are reused for the next detector
    if (e != cudaSuccess) { set_error("sky plan upload failed: %s", cudaGetErrorString(e)); delete pl; return SPIIR_ECUDA; }
    pl->n_tuples = std::max(pl->n_tuples, S.n_tuples);
  }
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) { set_error("device query failed: %s", cudaGetErrorString(e)); delete pl; return SPIIR_ECUDA; }
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

template <int D, int K, bool MAP>
static int sky_launch_one(const SkyParams& P, long long max_batches, int num_sms, size_t smem, cudaStream_t st) {
  static unsigned long long configured = 0;
  if (first_use_on_device(configured)) {
    SPIIR_CUDA_OK(cudaFuncSetAttribute(k_sky<D, K, MAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSkySmemMax));
  }
  const int grid = (int)std::max<long long>(1, std::min<long long>(max_batches, num_sms));
  k_sky<D, K, MAP><<<grid, kSkyThreads, smem, st>>>(P);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

template <int D, bool MAP>
static int sky_launch_k(int K, const SkyParams& P, long long max_pairs, int num_sms, size_t smem, cudaStream_t st) {
  const long long nb = (max_pairs + 32 * K - 1) / (32 * K);
  switch (K) {
    case 1: return sky_launch_one<D, 1, MAP>(P, nb, num_sms, smem, st);
    case 2: return sky_launch_one<D, 2, MAP>(P, nb, num_sms, smem, st);
    case 3: return sky_launch_one<D, 3, MAP>(P, nb, num_sms, smem, st);
    default: return sky_launch_one<D, 4, MAP>(P, nb, num_sms, smem, st);
  }
}

static int sky_run(spiir_sky_plan* pl, const spiir_snr_view* view, const spiir_trigger* trig, int32_t n_slots,
                   int32_t n_slides, int64_t step, const int32_t* mult, spiir_sky_result* out, float* map,
                   cudaStream_t st) {
  SPIIR_REQUIRE(pl && trig && out, "a pointer is NULL");
  if (int rcv = check_snr_view(view)) return rcv;
  SPIIR_REQUIRE(n_slots >= 0 && n_slots <= pl->max_slots, "n_slots %d exceeds the plan's max_slots %d", n_slots,
                pl->max_slots);
  if (int rcs = check_slides(n_slides, step, mult, pl->n_det)) return rcs;
  if (n_slots == 0) return SPIIR_OK;
  const int D = pl->n_det, S1 = n_slides > 0 ? n_slides : 1;
  int32_t* counts = (int32_t*)(pl->ws + pl->off_counts);
  SkyRec* lists = (SkyRec*)(pl->ws + pl->off_lists);
  SPIIR_CUDA_OK(cudaMemsetAsync(counts, 0, SPIIR_MAX_DET * 4, st));
  if (map) SPIIR_CUDA_OK(cudaMemsetAsync(map, 0, (size_t)n_slots * pl->n_pix * sizeof(float), st));
  k_sky_bin<<<(n_slots + 255) / 256, 256, 0, st>>>(trig, n_slots, D, S1, (const float2*)view->dev_z, view->det_stride,
                                                   view->row_stride, view->ring_len, view->k_newest, view->n_rows, lists, counts,
                                                   pl->max_slots, out);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  // pairs one launch can see at most (the real count is on the device): all slots of one detector
  const long long max_pairs = (long long)n_slots * S1;
  for (int T = 0; T < D; ++T) {
    const spiir_sky_stream& S = pl->st[T];
    SkyParams P;
    memset(&P, 0, sizeof(P));
    P.stream = (const float*)(pl->ws + S.off_slots); P.n_chunks = S.n_chunks;
    for (int wv = 0; wv <= kSkyWarps; ++wv) P.cb[wv] = S.cb[wv];
    P.n_pix = pl->n_pix;
    P.z = (const float2*)view->dev_z; P.det_stride = view->det_stride; P.row_stride = view->row_stride;
    P.ring_len = view->ring_len; P.k_newest = view->k_newest;
    P.trig = trig; P.list = lists + (size_t)T * pl->max_slots; P.counts = counts; P.T = T;
    P.n_slides = n_slides; P.step = step;
    for (int I = 0; I < D; ++I) {
      P.mult[I] = (mult && I != T) ? mult[I] : 0;
      P.lo[I] = S.lo[I]; P.W[I] = S.W[I]; P.woff[I] = S.woff[I];
    }
    // pairs per thread: as many as shared memory allows, fewer when the launch could not fill the SMs
    int K = S.k_max;
    while (K > 1 && max_pairs / D < (long long)pl->num_sms * 32 * K) --K;
    P.win_elems = sky_win_elems(S.ps, K);
    P.ps = S.ps;
    for (int I = 0; I < D; ++I) P.soff[I] = S.woff[I];
    // TMA bulk copies need 16-byte aligned sources: an aligned base and even strides (in complex samples)
    P.tma = (((uintptr_t)view->dev_z & 15) == 0 && view->det_stride % 2 == 0 && view->row_stride % 2 == 0 &&
             view->ring_len % 2 == 0) ? 1 : 0;
    P.out = out; P.map = map;
    const size_t smem = sky_smem_bytes(S.ps, pl->SW, K);
    int rc;
    if (D == 2)      rc = map ? sky_launch_k<2, true>(K, P, max_pairs, pl->num_sms, smem, st) : sky_launch_k<2, false>(K, P, max_pairs, pl->num_sms, smem, st);
    else if (D == 3) rc = map ? sky_launch_k<3, true>(K, P, max_pairs, pl->num_sms, smem, st) : sky_launch_k<3, false>(K, P, max_pairs, pl->num_sms, smem, st);
    else             rc = map ? sky_launch_k<4, true>(K, P, max_pairs, pl->num_sms, smem, st) : sky_launch_k<4, false>(K, P, max_pairs, pl->num_sms, smem, st);
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
