// Measurement helper: a dependency-free FP32 FFMA loop on every SM, so that bench.py
// can quote the ALU roofline measured in the same process and at the same clocks
// (the FP32 peak is not in MEASURED_PEAKS.json).
#include "spiir_internal.cuh"

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

extern "C" int spiir_fp32_peak_probe(int32_t reps, double* ms_out, double* fma_per_launch, void* stream) {
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
