// H5 / H6 for three detectors (the paper's H1-L1-V1 network, BASELINE.json configs 1, 3, 4) — the kernel that
// carries the benchmark's sky-search load.  Same arithmetic as k_sky in sky.cu (Eq. 28, PAPER.md:483:
// rho_c^2 = z^H (U I U^T) z as a quadratic form in the real products q = Re(z_I conj z_J)), re-organised
// around what the round-1 captures named as the losses (profiles/r1_ncu_summary.md §2, profiles/r2_*):
//
//   * The per-tuple refresh was 6 FP32 + 1 gather per pair every ~3.5 directions.  Of the five products that
//     involve the two other detectors, |z_f|^2 and Re(z_T conj z_f) depend on ONE window row only; they are
//     formed once per row when a batch is staged ("expanded" rows: A = |z_f|^2, B = Re(z_T conj z_f), re, im)
//     and the stream walks that detector fast.  A refresh is then two LDS.128 and one packed multiply-add
//     pair (the cross product with the slow detector) per TWO pairs.
//   * The slow detector's row changes ~8 times per warp and batch: its samples are read straight from the
//     ring through L2 (prefetched there when the batch is set up), so only the FAST detector's windows sit in
//     shared memory — the narrower of the two (43 rows for H1-L1).  That leaves room to land the NEXT batch's
//     raw windows (TMA bulk copies, completion on an mbarrier) while the current batch computes; the window
//     staging that was a fixed ~17 % per batch overlaps the main loop.
//   * Two pairs of a lane ("couple") are interleaved in shared memory so that a refresh loads packed
//     (pair a, pair b) operands directly: every FP32 instruction of the loop is a packed FMUL2 / FFMA2.
//
// The projector U2 U2^T has trace 2 (U2: orthonormal columns, Eq. 27), so M_TT = 2 - M_ss - M_ff and
//   rho_c^2 - 2 |z_T|^2 = M_ss (|z_s|^2 - |z_T|^2) + 2 M_Ts Re(z_T conj z_s) + M_ff (|z_f|^2 - |z_T|^2)
//                         + 2 M_Tf Re(z_T conj z_f) + 2 M_sf Re(z_s conj z_f):
// FIVE multiply-adds per direction and 20 bytes of weights; the constant 2 |z_T|^2 is added after the maximum.
//
// Stream (directions sorted by (slow row, fast row, pixel)), per chunk of 32 directions 896 bytes:
//   32 x float4 (w1 = M_ss, w2 = 2 M_Ts, w3 = M_ff, w4 = 2 M_Tf) | 32 x (w5 = 2 M_sf, control) | 32 x pixel
//   control: nref | fast row << 5 (its byte offset in a couple's block) | slow row << 16; nref = 0 same delay tuple as
//   the previous slot, 1 the fast row changed, 2 the slow row changed (refresh both; also the first slot of a warp's share).
//   The 16 + 8 byte split makes a slot two broadcast loads of 2 + 1 shared-memory wavefronts instead of 2 + 2.
#include <algorithm>
#include <climits>
#include <cstring>
#include <vector>

#include "sky_internal.cuh"

namespace spiir {

struct Sky3Params {
  const float* stream; int32_t n_chunks, n_pix;
  int16_t cb[kSkyWarps + 1];  // chunks [cb[w], cb[w+1]) of the stream are warp w's share (balanced by cost on the host)
  const float2* z; int64_t det_stride, row_stride, ring_len, k_newest;
  const SkyRec* list; const int32_t* counts;
  int32_t T, I_s, I_f;
  int32_t n_slides; int64_t step; int32_t mult_s, mult_f;
  int32_t lo_s, W_s, lo_f, W_f;
  int32_t fstride;            // bytes of a couple's block of expanded rows: 32 W_f + 16 (odd multiple of 16)
  int32_t rlen;               // float2 elements of one raw window in the landing area (even)
  int32_t tma;                // view is 16-byte friendly: stage with TMA bulk copies and prefetch into L2
  spiir_sky_result* out; float* map;
};

// Per pair, built when a batch is set up.  48 bytes.
struct __align__(16) Pair3 {
  const float2* zs;           // the slow detector's SNR row (element 0 of the ring)
  long long foff;             // element offset of the fast detector's SNR row in the view
  int32_t bs, bf;             // ring index of row 0 of the slow / fast window
  int32_t slot, slide, valid;
  int32_t sh;                 // 0/1: the raw fast window lands one sample late (TMA copies start 16-byte aligned)
  float2 vT;
};
static_assert(sizeof(Pair3) == 48, "Pair3 layout");

// Packed FP32 pairs are held as 64-bit values end to end (loaded as .b64, multiplied as .f32x2), so that a pair
// always sits in an aligned register pair: with float2 variables ptxas kept the halves apart and re-packed them
// with moves on every refresh.  Per component the roundings are those of __fmul_rn / __fmaf_rn.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
// one expanded row of a couple: (A0, A1), (B0, B1), (re0, re1), (im0, im1)
__device__ __forceinline__ void lds_row(uint32_t addr, f32x2& A, f32x2& B, f32x2& re, f32x2& im) {
  asm volatile("ld.shared.v2.b64 {%0, %1}, [%4];\n\tld.shared.v2.b64 {%2, %3}, [%4+16];"
               : "=l"(A), "=l"(B), "=l"(re), "=l"(im)
               : "r"(addr));
}

static int sky3_rlen(int W_f) { return (W_f + 3) & ~1; }
static int sky3_fstride(int W_f) { return 32 * W_f + 16; }
constexpr int kTileSlots = 3 * kSkyChunk + 2;   // a warp's ring of three stream chunks; slots 96, 97 mirror slots 0, 1
constexpr int kTileW4 = 0, kTileW2 = kTileSlots * 16, kTilePx = kTileW2 + kTileSlots * 8;   // byte offsets of the three arrays
constexpr int kTileBytes = (kTilePx + kTileSlots * 4 + 15) / 16 * 16;
constexpr int kTileWords = kTileBytes / 4;
constexpr int kChunkBytes = kSkyChunk * 28;     // a chunk of the stream in global memory
size_t sky3_smem_bytes(int W_f, int K) {
  const int NP = 32 * K;
  return (size_t)(NP / 2) * sky3_fstride(W_f) + (size_t)NP * sky3_rlen(W_f) * 8 + (size_t)kSkyWarps * kTileWords * 4 +
         (size_t)2 * NP * sizeof(Pair3) + (size_t)NP * sizeof(SkyRec) + (size_t)NP * 4;
}

template <int K, bool MAP>
__global__ void __launch_bounds__(kSkyThreads, 1) k_sky3(const __grid_constant__ Sky3Params P) {
  constexpr int NP = 32 * K, NC = NP / 2, KC = K / 2;
  static_assert(K % 2 == 0 && 2 * NP <= 256, "pairs come in couples; the merge reuses a warp's 256-word tile");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* Fb = smem_raw;                                                   // [NC] blocks of fstride bytes: expanded fast rows
  float2* R = reinterpret_cast<float2*>(Fb + (size_t)NC * P.fstride);             // [NP][rlen] raw windows of the NEXT batch
  float* tiles = reinterpret_cast<float*>(R + (size_t)NP * P.rlen);               // [warps][kTileWords]
  Pair3* pinfo = reinterpret_cast<Pair3*>(tiles + kSkyWarps * kTileWords);        // [2][NP]
  SkyRec* recbuf = reinterpret_cast<SkyRec*>(pinfo + 2 * NP);                     // [NP] records of the batch after the next
  int* wchunk = reinterpret_cast<int*>(recbuf + NP);                              // [NP] chunk holding each pair's maximum
  __shared__ uint64_t bar;                                                        // completion of a batch's TMA window copies

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int S1 = P.n_slides > 0 ? P.n_slides : 1;
  const long long n_pairs = (long long)P.counts[P.T] * S1;
  const long long n_batches = (n_pairs + NP - 1) / NP;
  const long long G = gridDim.x;
  if ((long long)blockIdx.x >= n_batches) return;
  const int64_t kmin = (P.k_newest - P.ring_len + 1 > 0) ? P.k_newest - P.ring_len + 1 : 0;
  float* mytile = tiles + warp * kTileWords;
  const int c_beg = P.cb[warp], c_end = P.cb[warp + 1];
  const uint32_t bar_a = sky_smem_u32(&bar);
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar_a), "r"(NP));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  uint32_t bar_phase = 0;

  // ---- pipeline stages -----------------------------------------------------------------------------------
  // (1) the 32-byte records of a batch -> recbuf, asynchronously (two 16-byte cp.async per pair)
  auto load_recs = [&](long long batch) {
    if (tid < NP) {
      const long long q = batch * NP + tid;
      if (q < n_pairs) {
        const SkyRec* src = P.list + q / S1;
        cp_async_16(recbuf + tid, src);
        cp_async_16(reinterpret_cast<char*>(recbuf + tid) + 16, reinterpret_cast<const char*>(src) + 16);
      }
    }
    cp_async_commit();
  };
  // (2) pair set-up: which trigger, which slide, is every gather inside the view, where the windows start
  auto build_pinfo = [&](long long batch, Pair3* pb) {
    if (tid < NP) {
      Pair3 pi;
      pi.zs = P.z; pi.foff = 0; pi.bs = 0; pi.bf = 0; pi.slot = -1; pi.slide = 0; pi.valid = 0; pi.sh = 0;
      pi.vT = make_float2(0.f, 0.f);
      const long long q = batch * NP + tid;
      if (q < n_pairs) {
        const SkyRec rc = recbuf[tid];
        pi.slot = rc.slot;
        pi.slide = (int)(q % S1) + (P.n_slides > 0 ? 1 : 0);
        const int64_t k0s = rc.k - (int64_t)pi.slide * P.step * P.mult_s + P.lo_s;
        const int64_t k0f = rc.k - (int64_t)pi.slide * P.step * P.mult_f + P.lo_f;
        const bool ok = rc.k_ok != 0 && k0s >= kmin && k0s + P.W_s - 1 <= P.k_newest && k0f >= kmin &&
                        k0f + P.W_f - 1 <= P.k_newest;
        if (ok) {
          pi.valid = 1;
          pi.vT = rc.vT;
          pi.zs = P.z + (size_t)P.I_s * P.det_stride + (size_t)rc.row * P.row_stride;
          pi.bs = (int32_t)(k0s % P.ring_len);
          // the fast window's first sample in the ring; TMA copies start at the 16-byte aligned sample at or before it
          const int64_t bf = k0f % P.ring_len;
          pi.sh = P.tma ? (int)(bf & 1) : 0;
          pi.foff = (long long)((size_t)P.I_f * P.det_stride + (size_t)rc.row * P.row_stride);
          pi.bf = (int32_t)bf;
        }
      }
      pb[tid] = pi;
    }
  };
  // (3) raw fast windows -> R (asynchronously); slow windows -> L2
  auto issue_windows = [&](const Pair3* pb) {
    if (P.tma) {
      if (tid < NP) {
        const Pair3 pi = pb[tid];
        if (pi.valid) {
          const float2* row = P.z + pi.foff;
          const int64_t idx0 = (int64_t)pi.bf - pi.sh;
          const int len = (P.W_f + pi.sh + 1) & ~1;                          // samples copied: even, covers the window
          const int n1 = (int)min((int64_t)len, P.ring_len - idx0);           // before the ring's end (even: ring_len is even)
          const uint32_t dst = sky_smem_u32(R + (size_t)tid * P.rlen);
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(len * 8) : "memory");
          tma_bulk_g2s(dst, row + idx0, (uint32_t)n1 * 8u, bar_a);
          if (n1 < len) tma_bulk_g2s(dst + (uint32_t)n1 * 8u, row, (uint32_t)(len - n1) * 8u, bar_a);
          // the slow window is read row by row from L2 during the main loop: ask for it now
          const int64_t s0 = (int64_t)pi.bs & ~(int64_t)1;
          const int slen = (P.W_s + 2) & ~1;
          const int m1 = (int)min((int64_t)slen, P.ring_len - s0);
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pi.zs + s0), "r"(m1 * 8) : "memory");
          if (m1 < slen) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pi.zs), "r"((slen - m1) * 8) : "memory");
        } else {
          asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar_a) : "memory");
        }
      }
    } else {
      for (int j = warp; j < NP; j += kSkyWarps) {
        const Pair3 pi = pb[j];
        if (!pi.valid) continue;
        const float2* row = P.z + pi.foff;
        float2* dst = R + (size_t)j * P.rlen;
        for (int r = lane; r < P.W_f; r += 32) {
          int64_t idx = (int64_t)pi.bf + r;
          if (idx >= P.ring_len) idx -= P.ring_len;
          cp_async_8(dst + r, row + idx);
        }
      }
      cp_async_commit();
    }
  };
  auto wait_windows = [&]() {
    if (P.tma) {
      mbar_wait_bounded(bar_a, bar_phase);
      bar_phase ^= 1u;
    } else {
      cp_async_wait_all();
      __syncthreads();
    }
  };
  // (4) R -> F: per couple and row (A0, A1, B0, B1 | re0, re1, im0, im1), A = |x|^2 - |z_T|^2, B = Re(z_T conj x); lanes take
  //     consecutive couples, whose blocks are an odd number of 16-byte units apart: conflict-free STS.128
  auto expand = [&](const Pair3* pb) {
    for (int t = tid; t < NC * P.W_f; t += kSkyThreads) {
      const int c = t % NC, r = t / NC;
      const int ja = (c & 31) + 64 * (c >> 5), jb = ja + 32;
      const Pair3* pa = pb + ja; const Pair3* pc = pb + jb;
      float2 xa = make_float2(0.f, 0.f), xb = make_float2(0.f, 0.f);
      if (pa->valid) xa = R[(size_t)ja * P.rlen + pa->sh + r];
      if (pc->valid) xb = R[(size_t)jb * P.rlen + pc->sh + r];
      const float2 va = pa->vT, vb = pc->vT;
      float4* dst = reinterpret_cast<float4*>(Fb + (size_t)c * P.fstride + (size_t)r * 32);
      dst[0] = make_float4(__fsub_rn(re_prod(xa, xa), re_prod(va, va)), __fsub_rn(re_prod(xb, xb), re_prod(vb, vb)),
                           re_prod(va, xa), re_prod(vb, xb));
      dst[1] = make_float4(xa.x, xb.x, xa.y, xb.y);
    }
  };

  // ---- prologue: the first batch up to its expanded windows, the records of the second
  long long b = blockIdx.x;
  load_recs(b);
  cp_async_wait_all();
  __syncthreads();
  build_pinfo(b, pinfo);
  __syncthreads();
  issue_windows(pinfo);
  if (b + G < n_batches) load_recs(b + G);
  wait_windows();
  expand(pinfo);
  int cur = 0;
  bool chunks_ahead = false;

  for (; b < n_batches; b += G) {
    const long long bn = b + G;
    const bool has_next = bn < n_batches;
    Pair3* pcur = pinfo + cur * NP;
    Pair3* pnxt = pinfo + (cur ^ 1) * NP;
    cp_async_wait_all();                               // the next batch's records have landed (and nothing else is pending)
    __syncthreads();                                   // ... for everyone; F and pinfo[cur] are complete
    if (has_next) {
      build_pinfo(bn, pnxt);
      __syncthreads();
      issue_windows(pnxt);                             // lands in R while this batch computes
      if (bn + G < n_batches) load_recs(bn + G);
    }
    // the warp's first two chunks of the direction stream -> its ring of three chunk buffers (cp.async, no registers)
    auto issue_chunk = [&](int c, int buf) {
      if (c < c_end) {
        const char* src = reinterpret_cast<const char*>(P.stream) + (size_t)c * kChunkBytes;
        char* t = reinterpret_cast<char*>(mytile);
        const int i = buf * kSkyChunk + lane;
        cp_async_16(t + kTileW4 + i * 16, src + lane * 16);
        cp_async_8(t + kTileW2 + i * 8, src + 512 + lane * 8);
        if (MAP) cp_async_4(t + kTilePx + i * 4, src + 768 + lane * 4);
        if (buf == 0 && lane < 2) {                    // slots 96, 97 mirror slots 0, 1: the look-ahead never wraps
          const int m = 3 * kSkyChunk + lane;
          cp_async_16(t + kTileW4 + m * 16, src + lane * 16);
          cp_async_8(t + kTileW2 + m * 8, src + 512 + lane * 8);
        }
      }
      cp_async_commit();
    };
    if (!chunks_ahead) {                               // first batch of this CTA: nothing was requested ahead
      __syncwarp();
      issue_chunk(c_beg, 1);
      issue_chunk(c_beg + 1, 2);
    }

    // ---- the direction stream: this warp's chunks
    f32x2 qp[KC][5];                                   // products of pairs (2i, 2i+1) side by side: packed FFMA2 operands
    f32x2 vsr[KC], vsi[KC];                            // the slow detector's sample of both pairs (re, re), (im, im)
    float best[K], seen[K]; int bch[K];
    long long mrow[K]; float q0m[K];                   // sky map only: row of the pair, its constant 2 |z_T|^2 term
    uint32_t fb[KC];
#pragma unroll
    for (int i = 0; i < KC; ++i) {
      fb[i] = sky_smem_u32(Fb + (size_t)(lane + 32 * i) * P.fstride);
      vsr[i] = pack2(0.f, 0.f); vsi[i] = pack2(0.f, 0.f);
#pragma unroll
      for (int e = 0; e < 5; ++e) qp[i][e] = pack2(0.f, 0.f);
    }
#pragma unroll
    for (int a = 0; a < K; ++a) {
      const Pair3* pp = pcur + lane + 32 * a;
      best[a] = -3.0e38f; seen[a] = -3.0e38f; bch[a] = c_beg;
      mrow[a] = (MAP && pp->valid) ? (long long)pp->slot * P.n_pix : -1;
      q0m[a] = MAP ? re_prod(pp->vT, pp->vT) : 0.f;
    }

    int rb = 1;                                        // ring buffer holding chunk ch (a batch starts in buffer 1)
    for (int ch = c_beg; ch < c_end; ++ch) {
      __syncwarp();                                    // every lane is done reading the buffer that is refilled now
      const int rb2 = rb >= 1 ? rb - 1 : 2;            // (rb + 2) % 3
      issue_chunk(ch + 2, rb2);
      cp_async_wait_group<1>();                        // chunks ch and ch + 1 have landed
      __syncwarp();
      // broadcast reads, two slots ahead of their use (the weights of a slot wait on nothing when it starts)
      const float4* w4p = reinterpret_cast<const float4*>(reinterpret_cast<const char*>(mytile) + kTileW4) + rb * kSkyChunk;
      const float2* w2p = reinterpret_cast<const float2*>(reinterpret_cast<const char*>(mytile) + kTileW2) + rb * kSkyChunk;
      const int* pxp = reinterpret_cast<const int*>(reinterpret_cast<const char*>(mytile) + kTilePx) + rb * kSkyChunk;
      float4 nA4 = w4p[0], nB4 = w4p[1];
      float2 nA2 = w2p[0], nB2 = w2p[1];
      rb = rb == 2 ? 0 : rb + 1;
      float pend[K];
#pragma unroll 4
      for (int s = 0; s < kSkyChunk; ++s) {
        const float4 w0 = nA4; const float2 w1 = nA2;
        nA4 = nB4; nA2 = nB2;
        nB4 = w4p[s + 2]; nB2 = w2p[s + 2];
        const int ctrl = __float_as_int(w1.y);
        if (ctrl & 3) {
          if (ctrl & 2) {
            // the slow detector's row changed: its sample from the ring (L2), the two products it enters alone
            const int rs = (ctrl >> 16) & ((1 << kSkyRowBits) - 1);
            float2 xs[K];
#pragma unroll
            for (int a = 0; a < K; ++a) {
              const Pair3* pp = pcur + lane + 32 * a;
              xs[a] = make_float2(0.f, 0.f);
              if (pp->valid) {
                long long e = (long long)pp->bs + rs;
                if (e >= P.ring_len) e -= P.ring_len;
                xs[a] = __ldg(pp->zs + e);
              }
            }
#pragma unroll
            for (int i = 0; i < KC; ++i) {
              const float2 va = pcur[lane + 64 * i].vT, vb = pcur[lane + 64 * i + 32].vT;
              const float2 xa = xs[2 * i], xb = xs[2 * i + 1];
              qp[i][0] = pack2(__fsub_rn(re_prod(xa, xa), re_prod(va, va)), __fsub_rn(re_prod(xb, xb), re_prod(vb, vb)));
              qp[i][1] = pack2(re_prod(va, xa), re_prod(vb, xb));
              vsr[i] = pack2(xa.x, xb.x); vsi[i] = pack2(xa.y, xb.y);
            }
          }
          // the fast row: A and B come expanded, the cross product with the slow sample is one packed multiply-add pair
          const uint32_t ro = (uint32_t)ctrl & 0x7fe0u;            // the fast row's byte offset, as stored
#pragma unroll
          for (int i = 0; i < KC; ++i) {
            f32x2 xre, xim;
            lds_row(fb[i] + ro, qp[i][2], qp[i][3], xre, xim);
            qp[i][4] = fma2(vsr[i], xre, mul2(vsi[i], xim));
          }
        }
        // the quadratic form of two pairs at a time: scalar weight x packed products
        float cval[K];
        const f32x2 ww[5] = {pack2(w0.x, w0.x), pack2(w0.y, w0.y), pack2(w0.z, w0.z), pack2(w0.w, w0.w), pack2(w1.x, w1.x)};
#pragma unroll
        for (int i = 0; i < KC; ++i) {
          f32x2 c2 = mul2(ww[0], qp[i][0]);
#pragma unroll
          for (int e = 1; e < 5; ++e) c2 = fma2(ww[e], qp[i][e], c2);
          unpack2(c2, cval[2 * i], cval[2 * i + 1]);
        }
#pragma unroll
        for (int a = 0; a < K; ++a) {
          if (MAP) {
            if (mrow[a] >= 0) P.map[mrow[a] + pxp[s]] = __fmaf_rn(2.f, q0m[a], cval[a]);
          }
          // two directions per maximum: the value of an even slot waits for its odd neighbour (one FMNMX3)
          if (s & 1) best[a] = fmax3(best[a], pend[a], cval[a]);
          else       pend[a] = cval[a];
        }
      }
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
    // the stream does not depend on the batch: the first two chunks of the next one are requested now (the merge is
    // done with the tiles) and land during the rescan and the staging of the next windows
    if (has_next) {
      issue_chunk(c_beg, 1);
      issue_chunk(c_beg + 1, 2);
    }
    chunks_ahead = has_next;
    // ---- a warp rescans the winning chunk of each of its 2 K pairs, lane = slot: every lane forms its own direction's
    //      products from scratch with the roundings of the staging and the main loop; the first lane holding the maximum
    //      gives the direction, tot2 and null2 there (Eq. 10)
    constexpr int PPW = NP / kSkyWarps, RB = (PPW % 8 == 0) ? 8 : ((PPW % 4 == 0) ? 4 : 2);   // requests in flight per round
    for (int u0 = 0; u0 < PPW; u0 += RB) {
      float4 wv4[RB]; float2 wv2[RB]; int wpx[RB]; float2 xs[RB];
#pragma unroll
      for (int u = 0; u < RB; ++u) {
        const int j = warp + (u0 + u) * kSkyWarps;
        const char* sp = reinterpret_cast<const char*>(P.stream) + (size_t)wchunk[j] * kChunkBytes;
        wv4[u] = __ldg(reinterpret_cast<const float4*>(sp) + lane);
        wv2[u] = __ldg(reinterpret_cast<const float2*>(sp + 512) + lane);
        wpx[u] = __ldg(reinterpret_cast<const int*>(sp + 768) + lane);
        const Pair3* pp = pcur + j;
        xs[u] = make_float2(0.f, 0.f);
        if (pp->valid) {
          const int rs = (__float_as_int(wv2[u].y) >> 16) & ((1 << kSkyRowBits) - 1);
          long long e = (long long)pp->bs + rs;
          if (e >= P.ring_len) e -= P.ring_len;
          xs[u] = __ldg(pp->zs + e);
        }
      }
#pragma unroll
      for (int u = 0; u < RB; ++u) {
        const int j = warp + (u0 + u) * kSkyWarps;
        const Pair3 pi = pcur[j];
        if (pi.slot < 0) continue;
        spiir_sky_result res; res.coh2 = 0.f; res.null2 = 0.f; res.tot2 = 0.f; res.pix = -1;
        if (pi.valid) {
          const float4 w0 = wv4[u];
          const int ctrl = __float_as_int(wv2[u].y);
          const int rf = (ctrl >> 5) & ((1 << kSkyRowBits) - 1);
          const int c = (j & 31) + 32 * (j >> 6), half = (j >> 5) & 1;
          const float* row = reinterpret_cast<const float*>(Fb + (size_t)c * P.fstride + (size_t)rf * 32);
          const float2 xf = make_float2(row[4 + half], row[6 + half]);
          const float q0 = re_prod(pi.vT, pi.vT), xs2 = re_prod(xs[u], xs[u]), xf2 = re_prod(xf, xf);
          const float q1 = __fsub_rn(xs2, q0), q2 = re_prod(pi.vT, xs[u]);
          const float q3 = __fsub_rn(xf2, q0), q4 = re_prod(pi.vT, xf), q5 = re_prod(xs[u], xf);
          const float tot = (q0 + xs2) + xf2;
          float cc = __fmul_rn(w0.x, q1);
          cc = __fmaf_rn(w0.y, q2, cc); cc = __fmaf_rn(w0.z, q3, cc); cc = __fmaf_rn(w0.w, q4, cc);
          cc = __fmaf_rn(wv2[u].x, q5, cc);
          float cm = cc;
#pragma unroll
          for (int o = 16; o; o >>= 1) cm = fmaxf(cm, __shfl_xor_sync(0xffffffffu, cm, o));
          const int src = __ffs(__ballot_sync(0xffffffffu, cc == cm)) - 1;
          res.coh2 = __fmaf_rn(2.f, q0, cm);
          res.tot2 = __shfl_sync(0xffffffffu, tot, src);
          res.pix = __shfl_sync(0xffffffffu, wpx[u], src);
          res.null2 = fmaxf(res.tot2 - res.coh2, 0.f);
        }
        if (lane == 0) P.out[(size_t)pi.slot * S1 + (P.n_slides > 0 ? pi.slide - 1 : 0)] = res;
      }
    }
    __syncthreads();                                   // F and pinfo[cur] are free
    if (has_next) {
      wait_windows();
      expand(pnxt);
    }
    cur ^= 1;
  }
}

// Builds the stream of trigger detector T in the three-detector format (host).
void sky3_build_stream(spiir_sky_plan* pl, int T, const float* u2, const int32_t* delay, std::vector<float>& slots) {
  const int D = 3, n_pix = pl->n_pix;
  spiir_sky_stream& S = pl->st[T];
  const int Is = S.I_s, If = S.I_f;
  std::vector<int32_t> rs(n_pix), rf(n_pix), order(n_pix);
  for (int p = 0; p < n_pix; ++p) {
    rs[p] = delay[(size_t)p * D + Is] - delay[(size_t)p * D + T] - S.lo[Is];
    rf[p] = delay[(size_t)p * D + If] - delay[(size_t)p * D + T] - S.lo[If];
    order[p] = p;
  }
  std::sort(order.begin(), order.end(), [&](int32_t x, int32_t y) {
    if (rs[x] != rs[y]) return rs[x] < rs[y];
    if (rf[x] != rf[y]) return rf[x] < rf[y];
    return x < y;
  });
  // what each slot refreshes, before the warps' shares are cut: 0 nothing, 1 the fast row, 2 both
  const int n_chunks = pl->cap_slots / kSkyChunk;
  std::vector<int> nr(pl->cap_slots, 0);
  S.n_tuples = 0;
  for (int r = 0; r < n_pix; ++r) {
    const int p = order[r];
    nr[r] = 2;
    if (r > 0) {
      const int pp = order[r - 1];
      nr[r] = rs[pp] != rs[p] ? 2 : (rf[pp] != rf[p] ? 1 : 0);
    }
    if (nr[r]) ++S.n_tuples;
  }
  // the 16 warps take contiguous runs of chunks of about equal COST (a refresh costs about as much as one and a
  // half directions, a slow-row change as much as eight: it waits on L2): without this the warps whose share is
  // dense in delay tuples finish last and the others idle at the barrier (3.5 % of the kernel, profiles/r2)
  {
    std::vector<double> cost(n_chunks, 0.0);
    double total = 0;
    for (int c = 0; c < n_chunks; ++c) {
      double x = kSkyChunk;
      for (int r = c * kSkyChunk; r < (c + 1) * kSkyChunk; ++r) x += nr[r] == 2 ? 8.0 : (nr[r] == 1 ? 1.5 : 0.0);
      cost[c] = x; total += x;
    }
    double acc = 0; int w = 1;
    S.cb[0] = 0;
    for (int c = 0; c < n_chunks && w < kSkyWarps; ++c) {
      acc += cost[c];
      if (acc >= total * w / kSkyWarps) S.cb[w++] = (int16_t)(c + 1);
    }
    for (; w <= kSkyWarps; ++w) S.cb[w] = (int16_t)n_chunks;
  }
  slots.assign((size_t)pl->cap_slots * 7, 0.f);        // 28 bytes per direction, chunk by chunk (layout above)
  int last_ctrl = 0; float last_w[5] = {0, 0, 0, 0, 0}; int32_t last_pix = 0;
  for (int r = 0; r < pl->cap_slots; ++r) {
    float* cbase = &slots[(size_t)(r / kSkyChunk) * (kChunkBytes / 4)];
    const int l = r % kSkyChunk;
    float* w4 = cbase + l * 4; float* w2 = cbase + 128 + l * 2; float* px = cbase + 192 + l;
    if (r < n_pix) {
      const int p = order[r];
      int nref = nr[r];
      for (int wv = 0; wv < kSkyWarps; ++wv)
        if (r == S.cb[wv] * kSkyChunk) nref = 2;   // a warp's share of the stream starts from nothing
      const float* u = u2 + (size_t)p * D * 2;
      auto M = [&](int I, int J) { return (double)u[2 * I] * u[2 * J] + (double)u[2 * I + 1] * u[2 * J + 1]; };
      // projector U2 U2^T in float64 from the float32 table, rounded once, in the kernel's order; its trace must be 2
      const double tr = M(T, T) + M(Is, Is) + M(If, If);
      if (!(tr > 2.0 - 1e-4 && tr < 2.0 + 1e-4)) S.bad_trace = 1;
      last_w[0] = (float)M(Is, Is);
      last_w[1] = (float)(2.0 * M(T, Is));
      last_w[2] = (float)M(If, If);
      last_w[3] = (float)(2.0 * M(T, If));
      last_w[4] = (float)(2.0 * M(Is, If));
      last_pix = p;
      last_ctrl = nref | (rf[p] << 5) | (rs[p] << 16);
    } else {
      last_ctrl &= ~3;                       // padding: the last direction again, nothing to refresh
    }
    w4[0] = last_w[0]; w4[1] = last_w[1]; w4[2] = last_w[2]; w4[3] = last_w[3];
    w2[0] = last_w[4];
    memcpy(w2 + 1, &last_ctrl, 4);
    memcpy(px, &last_pix, 4);
    if (r < n_pix) last_ctrl &= ~3;
  }
  S.n_chunks = pl->cap_slots / kSkyChunk;
}

template <int K, bool MAP>
static int sky3_launch_one(const Sky3Params& P, long long max_batches, int num_sms, size_t smem, cudaStream_t st) {
  static unsigned long long configured = 0;
  if (first_use_on_device(configured)) {
    SPIIR_CUDA_OK(cudaFuncSetAttribute(k_sky3<K, MAP>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSkySmemMax));
  }
  const int grid = (int)std::max<long long>(1, std::min<long long>(max_batches, num_sms));
  k_sky3<K, MAP><<<grid, kSkyThreads, smem, st>>>(P);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

int sky3_launch(const spiir_sky_plan* pl, int T, const spiir_snr_view* view, const SkyRec* list, const int32_t* counts,
                long long max_pairs, int32_t n_slides, int64_t step, const int32_t* mult, spiir_sky_result* out, float* map,
                cudaStream_t st) {
  const spiir_sky_stream& S = pl->st[T];
  Sky3Params P;
  memset(&P, 0, sizeof(P));
  P.stream = (const float*)(pl->ws + S.off_slots); P.n_chunks = S.n_chunks;
  for (int w = 0; w <= kSkyWarps; ++w) P.cb[w] = S.cb[w];
  P.n_pix = pl->n_pix;
  P.z = (const float2*)view->dev_z; P.det_stride = view->det_stride; P.row_stride = view->row_stride;
  P.ring_len = view->ring_len; P.k_newest = view->k_newest;
  P.list = list; P.counts = counts;
  P.T = T; P.I_s = S.I_s; P.I_f = S.I_f;
  P.n_slides = n_slides; P.step = step;
  P.mult_s = mult ? mult[S.I_s] : 0; P.mult_f = mult ? mult[S.I_f] : 0;
  P.lo_s = S.lo[S.I_s]; P.W_s = S.W[S.I_s]; P.lo_f = S.lo[S.I_f]; P.W_f = S.W[S.I_f];
  P.fstride = sky3_fstride(P.W_f); P.rlen = sky3_rlen(P.W_f);
  // TMA bulk copies need 16-byte aligned sources: an aligned base and even strides (in complex samples)
  P.tma = (((uintptr_t)view->dev_z & 15) == 0 && view->det_stride % 2 == 0 && view->row_stride % 2 == 0 &&
           view->ring_len % 2 == 0) ? 1 : 0;
  P.out = out; P.map = map;
  // pairs per thread: as many as shared memory allows, fewer when the launch could not fill the SMs
  int K = S.k3;
  while (K > 2 && max_pairs / 3 < (long long)pl->num_sms * 32 * K) K -= 2;
  const size_t smem = sky3_smem_bytes(P.W_f, K);
  const long long nb = (max_pairs + 32 * K - 1) / (32 * K);
  if (K >= 4) return map ? sky3_launch_one<4, true>(P, nb, pl->num_sms, smem, st) : sky3_launch_one<4, false>(P, nb, pl->num_sms, smem, st);
  return map ? sky3_launch_one<2, true>(P, nb, pl->num_sms, smem, st) : sky3_launch_one<2, false>(P, nb, pl->num_sms, smem, st);
}

}  // namespace spiir
