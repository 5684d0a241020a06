// H4 — per-second candidate selection on the device.
//
//   mode 0  one candidate per (detector, template): the sample of largest |z|^2 in
//           the last chunk.  The arg-max itself is fused into k_combine (it sees every
//           output sample anyway); this file only turns its records into trigger slots.
//   mode 1  the paper's two-step rule per bank of `bank_size` templates: (i) at each
//           sample the loudest template of the bank, kept iff above threshold;
//           (ii) per template the loudest kept sample.  Step (ii) is a 64-bit
//           atomicMax on key = (|z|^2 bits << 32) | (0xFFFFFFFF - k): larger |z|^2
//           wins, then the lower k — deterministic whatever the thread order.
//
// |z|^2 is decided in float32 as fl(fl(re*re) + fl(im*im)) (spiir.h).
#include "spiir_internal.cuh"

namespace spiir {

constexpr int kPeakThreads = 256;

__device__ __forceinline__ float mag2_rn(float2 z) {
  return __fadd_rn(__fmul_rn(z.x, z.x), __fmul_rn(z.y, z.y));
}

__device__ __forceinline__ void count_valid(bool valid, int32_t* count) {
  const unsigned m = __ballot_sync(0xffffffffu, valid);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(count, __popc(m));
}

__global__ void __launch_bounds__(kPeakThreads) k_peaks_mode0(const PeakParams p) {
  const int i = blockIdx.x * kPeakThreads + threadIdx.x;
  bool valid = false;
  if (i < p.D * p.T) {
    const PeakRec r = p.peak[i];
    valid = r.m2 > p.thr2;
    spiir_trigger t;
    t.valid = valid ? 1 : 0; t.tmpl = i % p.T; t.det = i / p.T; t._pad = 0;
    t.k = r.k; t.z_re = r.zr; t.z_im = r.zi; t.snr = sqrtf(r.m2); t._pad2 = 0.f;
    p.trig[i] = t;
  }
  count_valid(valid, p.count);
}

// step (i): thread = one output sample of one (detector, bank)
__global__ void __launch_bounds__(kPeakThreads) k_peaks_m1_scan(const PeakParams p) {
  const int k = blockIdx.x * kPeakThreads + threadIdx.x;
  const int bank = blockIdx.y, det = blockIdx.z;
  if (k >= p.n) return;
  const int t0 = bank * p.bank_size, t1 = min(p.T, t0 + p.bank_size);
  const int64_t col = (p.k0 + k) % p.ring_len;
  const float2* z = p.ring + (size_t)det * p.ring_det_stride + col;
  float bm = -1.f; int ts = t0;
  for (int t = t0; t < t1; ++t) {
    const float m2 = mag2_rn(z[(size_t)t * p.ring_len]);
    if (m2 > bm) { bm = m2; ts = t; }
  }
  if (bm > p.thr2) {
    const unsigned long long key =
        ((unsigned long long)__float_as_uint(bm) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)k);
    atomicMax(p.key + (size_t)det * p.T + ts, key);
  }
}

// step (ii) has happened in the atomics; decode the keys into trigger slots
__global__ void __launch_bounds__(kPeakThreads) k_peaks_m1_final(const PeakParams p) {
  const int i = blockIdx.x * kPeakThreads + threadIdx.x;
  bool valid = false;
  if (i < p.D * p.T) {
    const unsigned long long key = p.key[i];
    valid = key != 0ull;
    spiir_trigger t;
    t.valid = valid ? 1 : 0; t.tmpl = i % p.T; t.det = i / p.T; t._pad = 0; t._pad2 = 0.f;
    t.k = 0; t.z_re = 0.f; t.z_im = 0.f; t.snr = 0.f;
    if (valid) {
      const int k = (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull));
      const float m2 = __uint_as_float((unsigned)(key >> 32));
      const float2 z = p.ring[(size_t)t.det * p.ring_det_stride + (size_t)t.tmpl * p.ring_len +
                              (size_t)((p.k0 + k) % p.ring_len)];
      t.k = p.k0 + k; t.z_re = z.x; t.z_im = z.y; t.snr = sqrtf(m2);
    }
    p.trig[i] = t;
  }
  count_valid(valid, p.count);
}

int launch_peaks(const PeakParams& p, int mode, cudaStream_t st) {
  SPIIR_CUDA_OK(cudaMemsetAsync(p.count, 0, sizeof(int32_t), st));
  const int nslots = p.D * p.T;
  const int gslots = (nslots + kPeakThreads - 1) / kPeakThreads;
  if (mode == 0) {
    k_peaks_mode0<<<gslots, kPeakThreads, 0, st>>>(p);
    count_launch();
  } else {
    SPIIR_CUDA_OK(cudaMemsetAsync(p.key, 0, (size_t)nslots * sizeof(unsigned long long), st));
    const int n_banks = (p.T + p.bank_size - 1) / p.bank_size;
    k_peaks_m1_scan<<<dim3((p.n + kPeakThreads - 1) / kPeakThreads, n_banks, p.D), kPeakThreads, 0, st>>>(p);
    k_peaks_m1_final<<<gslots, kPeakThreads, 0, st>>>(p);
    count_launch(2);
  }
  SPIIR_CUDA_OK(cudaGetLastError());
  return SPIIR_OK;
}

}  // namespace spiir
