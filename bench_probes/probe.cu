// Measurement helpers of bench.py — NOT part of the product library (libspiir_b200.so allocates nothing and
// exports only the method's calls).  Built by bench_probes/build.py into bench_probes/libspiir_probe.so.
//   probe_fp32_peak: a dependency-free FP32 FFMA loop on every SM, so that bench.py can quote the ALU roofline
//   measured in the same process and at the same clocks (the FP32 peak is not in MEASURED_PEAKS.json).
#include <cuda_runtime.h>
#include <stdint.h>

#define SPIIR_OK 0
#define SPIIR_REQUIRE(cond, msg) do { if (!(cond)) return -1; } while (0)
#define SPIIR_CUDA_OK(expr) do { if ((expr) != cudaSuccess) return -3; } while (0)

namespace spiir {

constexpr int kProbeThreads = 256;
constexpr int kProbeChains = 16;
constexpr int kProbeIters = 4096;

__global__ void __launch_bounds__(kProbeThreads) k_fp32_probe(float* sink, float a, float b) {
  float v[kProbeChains];
#pragma unroll
  for (int c = 0; c < kProbeChains; ++c) v[c] = (float)(threadIdx.x + c) * 1e-3f;
  for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) v[c] = fmaf(v[c], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < kProbeChains; ++c) s += v[c];
  if (s == 123.456f) sink[0] = s;                  // never true; keeps the loop alive
}

}  // namespace spiir

extern "C" int probe_fp32_peak(int32_t reps, double* ms_out, double* fma_per_launch, void* stream) {
  using namespace spiir;
  SPIIR_REQUIRE(reps >= 1 && ms_out && fma_per_launch, "bad arguments");
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  SPIIR_CUDA_OK(cudaGetDevice(&dev));
  SPIIR_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  float* sink = nullptr;
  SPIIR_CUDA_OK(cudaMalloc(&sink, 4));               // measurement helper only; not on the hot path
  const int grid = sms * 8;
  cudaEvent_t e0, e1;
  SPIIR_CUDA_OK(cudaEventCreate(&e0));
  SPIIR_CUDA_OK(cudaEventCreate(&e1));
  k_fp32_probe<<<grid, kProbeThreads, 0, st>>>(sink, 0.999f, 1e-3f);   // warm-up
  SPIIR_CUDA_OK(cudaEventRecord(e0, st));
  for (int r = 0; r < reps; ++r) k_fp32_probe<<<grid, kProbeThreads, 0, st>>>(sink, 0.999f, 1e-3f);
  SPIIR_CUDA_OK(cudaEventRecord(e1, st));
  SPIIR_CUDA_OK(cudaEventSynchronize(e1));
  float ms = 0.f;
  SPIIR_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  *ms_out = ms;
  *fma_per_launch = (double)grid * kProbeThreads * kProbeChains * (double)kProbeIters;
  return SPIIR_OK;
}

// ------------------------------------------------------------------------------------------------
// Pipe probes behind DESIGN.md §6: register-only copies of the two hot inner loops, so that bench.py
// can quote, from committed code and in the same process, what the FP32 pipe gives each operation mix.
//   mode 1  the recursion of k_bank (F = 11 filters per lane, 4 samples per iteration: FMUL, 2 FFMA
//           and one FADD per component and update = 8 lane-operations), 2 CTAs of 256 threads per SM
//   mode 2  the quadratic form of k_sky as packed FFMA2 with vector-register operands (6 lane-operations
//           per evaluation, 2 evaluations per instruction), one CTA of 512 threads per SM
//   mode 3  the same quadratic form as scalar FFMA
namespace spiir {

constexpr int kPF = 11, kPIt = 2048;

__global__ void __launch_bounds__(256, 2) k_probe_recursion(const float4* coef, float* sink) {
  float ar[kPF], ai[kPF], br[kPF], bi[kPF], yr[kPF], yi[kPF];
#pragma unroll
  for (int f = 0; f < kPF; ++f) {
    const float4 c = coef[f * 256 + threadIdx.x];
    ar[f] = c.x; ai[f] = c.y; br[f] = c.z; bi[f] = c.w; yr[f] = 0.f; yi[f] = 0.f;
  }
  float acc = 0.f, x0 = sink[1 + (threadIdx.x & 7)];
  for (int it = 0; it < kPIt; ++it) {
    float s[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) s[q] = 0.f;
#pragma unroll
    for (int f = 0; f < kPF; ++f) {
      float a = yr[f], b = yi[f];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float xq = x0 + (float)q;
        const float tr = fmaf(-ai[f], b, br[f] * xq), ti = fmaf(ai[f], a, bi[f] * xq);
        const float nr = fmaf(ar[f], a, tr), ni = fmaf(ar[f], b, ti);
        a = nr; b = ni;
        s[2 * q] += nr; s[2 * q + 1] += ni;
      }
      yr[f] = a; yi[f] = b;
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) acc += s[q];
    x0 *= 0.999f;
  }
  if (acc == 123.456f) sink[0] = acc;
#pragma unroll
  for (int f = 0; f < kPF; ++f)
    if (yr[f] == 77.7f) sink[0] = yi[f];
}

constexpr int kPCh = 4;
template <bool PACKED>
__global__ void __launch_bounds__(512, 1) k_probe_quadform(const float* wts, float* sink) {
  float2 q[kPCh][6], best[kPCh];
#pragma unroll
  for (int c = 0; c < kPCh; ++c) {
    best[c] = make_float2(-1.f, -1.f);
#pragma unroll
    for (int e = 0; e < 6; ++e) q[c][e] = make_float2(sink[1 + ((c + e + threadIdx.x) & 7)], sink[1 + ((c + e + 1) & 7)]);
  }
  float w[6];
#pragma unroll
  for (int e = 0; e < 6; ++e) w[e] = wts[e + (threadIdx.x & 1)];
  for (int it = 0; it < kPIt; ++it) {
#pragma unroll
    for (int c = 0; c < kPCh; ++c) {
      float2 a;
      if (PACKED) {
        a = __fmul2_rn(make_float2(w[0], w[0]), q[c][0]);
#pragma unroll
        for (int e = 1; e < 6; ++e) a = __ffma2_rn(make_float2(w[e], w[e]), q[c][e], a);
      } else {
        a.x = w[0] * q[c][0].x; a.y = w[0] * q[c][0].y;
#pragma unroll
        for (int e = 1; e < 6; ++e) { a.x = fmaf(w[e], q[c][e].x, a.x); a.y = fmaf(w[e], q[c][e].y, a.y); }
      }
      best[c].x = fmaxf(best[c].x, a.x); best[c].y = fmaxf(best[c].y, a.y);
    }
#pragma unroll
    for (int e = 0; e < 6; ++e) w[e] *= 1.0001f;
  }
  float s = 0.f;
#pragma unroll
  for (int c = 0; c < kPCh; ++c) s += best[c].x + best[c].y;
  if (s == 123.456f) sink[0] = s;
}

}  // namespace spiir

extern "C" int probe_pipe(int32_t mode, int32_t reps, double* ms_out, double* lane_ops_per_launch, void* stream) {
  using namespace spiir;
  SPIIR_REQUIRE(mode >= 1 && mode <= 3 && reps >= 1 && ms_out && lane_ops_per_launch, "bad arguments");
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  SPIIR_CUDA_OK(cudaGetDevice(&dev));
  SPIIR_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  float* buf = nullptr;                
  const size_t n_coef = (size_t)kPF * 256 * 4;
  SPIIR_CUDA_OK(cudaMalloc(&buf, (16 + n_coef) * sizeof(float)));
  SPIIR_CUDA_OK(cudaMemsetAsync(buf, 0, (16 + n_coef) * sizeof(float), st));
  cudaEvent_t e0, e1;
  SPIIR_CUDA_OK(cudaEventCreate(&e0));
  SPIIR_CUDA_OK(cudaEventCreate(&e1));
  double ops = 0;
  for (int r = -1; r < reps; ++r) {                      // r = -1: warm-up
    if (r == 0) SPIIR_CUDA_OK(cudaEventRecord(e0, st));
    if (mode == 1) {
      k_probe_recursion<<<sms * 2, 256, 0, st>>>(reinterpret_cast<const float4*>(buf + 16), buf);
      ops = (double)sms * 2 * 256 * kPF * 4 * kPIt * 8.0;
    } else if (mode == 2) {
      k_probe_quadform<true><<<sms, 512, 0, st>>>(buf + 1, buf);
      ops = (double)sms * 512 * kPCh * 2 * kPIt * 6.0;
    } else {
      k_probe_quadform<false><<<sms, 512, 0, st>>>(buf + 1, buf);
      ops = (double)sms * 512 * kPCh * 2 * kPIt * 6.0;
    }
  }
  SPIIR_CUDA_OK(cudaEventRecord(e1, st));
  SPIIR_CUDA_OK(cudaEventSynchronize(e1));
  float ms = 0.f;
  SPIIR_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(buf);
  *ms_out = ms;
  *lane_ops_per_launch = ops;
  return SPIIR_OK;
}
