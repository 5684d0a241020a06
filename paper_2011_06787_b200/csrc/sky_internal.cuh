// Declarations of the sky search (sky.cu: plan, binning, the N_d = 2..4 kernel) that other translation units may
// need.  Nothing here is visible through include/spiir.h.
#pragma once
#include "spiir_internal.cuh"

namespace spiir {

constexpr int kSkyThreads = 512;
constexpr int kSkyWarps = kSkyThreads / 32;
constexpr int kSkyChunk = 32;               // slots per stream chunk (one per lane when staging)
constexpr int kSkySmemMax = 226 * 1024;     // opt-in dynamic shared memory per CTA on sm_100 (227 KB) less the static part
constexpr int kSkyRowBits = 10;             // bits of a window row in a slot's control word

// One candidate as k_sky_bin leaves it for the search kernels: everything a (candidate, slide) pair needs
// from the trigger and the trigger detector's SNR in ONE 32-byte read (the chain list -> trigger -> z would
// be three dependent HBM latencies at the head of every batch, and z_T the same for all slides).
struct __align__(16) SkyRec {
  int32_t slot, row;
  int64_t k;
  float2 vT;                  // z_T(row, k); zero when k is outside the view
  int32_t k_ok, _pad;
};

// ---- PTX helpers
__device__ __forceinline__ uint32_t sky_smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ void cp_async_8(void* dst_smem, const void* src_gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sky_smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_4(void* dst_smem, const void* src_gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sky_smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_16(void* dst_smem, const void* src_gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sky_smem_u32(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ float2 lds64(uint32_t addr) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
  return v;
}
// max of three (one FMNMX3 on sm_100; the same NaN rule as fmaxf)
__device__ __forceinline__ float fmax3(float a, float b, float c) {
  float r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
  return r;
}
// q_IJ = Re(v_I conj v_J), the same two roundings wherever it is formed (staging, main loop and rescan)
__device__ __forceinline__ float re_prod(float2 x, float2 y) { return __fmaf_rn(x.x, y.x, __fmul_rn(x.y, y.y)); }

// Waits for the phase `parity` of an mbarrier.  try_wait suspends the thread for a hardware time slice per
// poll; a copy that faulted or an expect_tx that disagrees with the bytes issued would otherwise spin forever,
// so the wait is bounded (seconds) and traps: the launch then fails with an error instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait_bounded(uint32_t bar_addr, uint32_t parity) {
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
        : "r"(bar_addr), "r"(parity)
        : "memory");
    if (done) return;
  }
  __trap();
}
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst_smem, const void* src_gmem, uint32_t bytes, uint32_t bar_addr) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
               "l"(src_gmem), "r"(bytes), "r"(bar_addr)
               : "memory");
}

}  // namespace spiir

struct spiir_sky_stream {                 // the direction stream of one trigger detector
  int n_chunks = 0, n_tuples = 0, rows = 0, k_max = 0;
  int lo[SPIIR_MAX_DET], W[SPIIR_MAX_DET], woff[SPIIR_MAX_DET];   // woff: offset of the detector's segment in a pair's block
  int ps = 0;                             // float2 elements of a pair's block (even)
  size_t off_slots = 0;
  int bad_trace = 0;                      // set by the stream builders when U2 U2^T does not have trace 2
  int32_t cb[17] = {0};                   // chunk boundaries of the 16 warps' shares, balanced by cost (any n_pix: 32-bit)
};

struct spiir_sky_plan {
  int n_det = 0, n_pix = 0, max_slots = 0, n_tuples = 0, SW = 0, cap_slots = 0;
  char* ws = nullptr;
  size_t off_lists = 0, off_counts = 0, bytes = 0;
  spiir_sky_stream st[SPIIR_MAX_DET];
  int num_sms = 148;
};
