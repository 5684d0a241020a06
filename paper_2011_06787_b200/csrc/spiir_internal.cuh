// Internal declarations shared by the translation units of libspiir_b200.so.
// Nothing here is visible through include/spiir.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>

#include "../../include/spiir.h"

namespace spiir {

void set_error(const char* fmt, ...);
void count_launch(int n = 1);

// Function attributes (opt-in shared memory) are per device: true the first time a launch site runs on
// the current device.
inline bool first_use_on_device(unsigned long long& mask) {
  int dev = 0;
  cudaGetDevice(&dev);
  const unsigned long long bit = 1ull << (dev & 63);
  if (mask & bit) return false;
  mask |= bit;
  return true;
}

#define SPIIR_CUDA_OK(expr)                                                         \
  do {                                                                              \
    cudaError_t e_ = (expr);                                                        \
    if (e_ != cudaSuccess) {                                                        \
      spiir::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_),      \
                       __FILE__, __LINE__);                                         \
      return SPIIR_ECUDA;                                                           \
    }                                                                               \
  } while (0)

#define SPIIR_REQUIRE(cond, ...)                                                    \
  do {                                                                              \
    if (!(cond)) {                                                                  \
      spiir::set_error(__VA_ARGS__);                                                \
      return SPIIR_EINVAL;                                                          \
    }                                                                               \
  } while (0)

// A caller's spiir_snr_view, checked the same way by every entry point that takes one.  n_rows joined the struct
// after its first five fields: a caller that fills only those on an uninitialised struct passes garbage there, and a
// huge value would switch off the kernels' row test.  A trigger's tmpl is an int32, so no honest view has more rows
// than that; strides are element counts and cannot be negative.  (No bound ties n_rows to det_stride: detector-
// interleaved layouts with det_stride < row_stride are legitimate.)
inline int check_snr_view(const spiir_snr_view* v) {
  SPIIR_REQUIRE(v != nullptr, "view is NULL");
  SPIIR_REQUIRE(v->dev_z != nullptr, "view: dev_z is NULL");
  SPIIR_REQUIRE(v->ring_len >= 1, "view: ring_len %lld < 1", (long long)v->ring_len);
  SPIIR_REQUIRE(v->n_rows >= 1 && v->n_rows <= 0x7fffffffLL,
                "view: n_rows %lld outside 1..2^31-1 (zero-initialise spiir_snr_view and set every field)",
                (long long)v->n_rows);
  SPIIR_REQUIRE(v->det_stride >= 0 && v->row_stride >= 0, "view: negative stride");
  return SPIIR_OK;
}

// Time-slide arguments common to the background search, xi^2 on slides and the slid windows:
// the largest shift n_slides * step * |mult| must stay far inside int64 (2^40 samples is 17 years at 2048 Hz).
inline int check_slides(int32_t n_slides, int64_t step, const int32_t* mult, int32_t n_det) {
  SPIIR_REQUIRE(n_slides >= 0, "n_slides < 0");
  if (n_slides == 0) return SPIIR_OK;
  SPIIR_REQUIRE(mult != nullptr && step >= 0, "time slides need host_slide_mult and step >= 0");
  SPIIR_REQUIRE(step <= (1ll << 40), "step_samples %lld is beyond 2^40", (long long)step);
  for (int I = 0; I < n_det; ++I) {
    const long long m = mult[I] < 0 ? -(long long)mult[I] : (long long)mult[I];
    SPIIR_REQUIRE(m == 0 || step == 0 || (long long)n_slides * m <= (1ll << 40) / step,
                  "slide shift n_slides * step_samples * |host_slide_mult[%d]| is beyond 2^40 samples", I);
  }
  return SPIIR_OK;
}

constexpr int kReplicas = 4;        // pre-shifted copies of each band's input (aligned LDS.128 for any delay)
constexpr int kReplicas2 = 8;       // ... in a band whose launch is bound by shared-memory conflicts: copy r + 4 gives every
                                    // filter a second choice of 16-byte bank group (bank.cu, placement)
constexpr int kBankThreads = 256;   // threads per CTA of the recursion kernel
constexpr int kBankWarps = kBankThreads / 32;
constexpr int kSubChunkMax = 2048;  // samples of one band staged in shared memory at a time
constexpr int kUpHist = 15;         // interpolator history: 16 non-zero taps per output parity
constexpr int kSmemFloatsMax = 6400;  // per replica: Hs + sub-chunk <= this (4 replicas -> 100 KB)

// Device-side description of one rate band, passed by value inside BankParams.
struct BandDev {
  const float4* coef;     // [wu][F][32]  (a.re, a.im, b.re, b.im); two-sample (odd-only) band: (a^2.re, a^2.im, b.re, b.im)
  const float2* coef2;    // [wu][F][32]  two-sample band only: a b
  const int32_t* off;     // [wu][F][32]  float offset of the filter's first sample in the replica set
  float2* state;          // [det][wu][F][32]
  float2* S;              // [det][unit][nmax] per-unit partial band sums of the current chunk
  const float* xrep;      // current-parity replica set of detector 0: [rep][cap]
  int64_t x_det_stride;   // floats between detectors in xrep
  int64_t state_det_stride, S_det_stride;   // elements
  int32_t n;              // samples of this band in the current chunk
  int32_t nmax;           // capacity (samples per chunk)
  int32_t Hcap, Hs;       // global / shared history depth, multiples of 4
  int32_t cap;            // floats per replica in global memory
  int32_t reps;           // floats per replica in shared memory ( = Hs + sub-chunk capacity )
  int32_t nsub;           // sub-chunk length for this call
  int32_t odd;            // 1: only odd samples are summed and stored, S[..][m] = s[2m+1] (band above the output rate)
  int32_t nrep, pad;      // replicas of this band (4 or 8); samples of extra history in front of a staged row (0 or 4)
};

struct BankParams {
  BandDev band[SPIIR_MAX_BANDS];
};

struct CtaWork { int32_t band, wu_begin, wu_end, xg; };   // xg: long-delay units, input read from global memory

// Kernel parameter blocks (bank_kernels.cu), filled by the host code in bank.cu.
struct PrepParams {
  const float* strain;     // [n_det][n0]
  int32_t n0, n_bands;
  float* xnew[SPIIR_MAX_BANDS];        // replica 0 of detector 0, new parity
  const float* xold[SPIIR_MAX_BANDS];  // replica 0 of detector 0, old parity
  int64_t x_det_stride[SPIIR_MAX_BANDS];
  int32_t cap[SPIIR_MAX_BANDS], Hcap[SPIIR_MAX_BANDS], n[SPIIR_MAX_BANDS], prev_n[SPIIR_MAX_BANDS], nrep[SPIIR_MAX_BANDS];
  const float* taps_dec;   // device [32]
};

struct PeakRec { long long k; float zr, zi, m2; int32_t _pad; };

struct CombineParams {
  const float2* S[SPIIR_MAX_BANDS];
  int64_t S_det_stride[SPIIR_MAX_BANDS];
  int32_t nmax[SPIIR_MAX_BANDS], n[SPIIR_MAX_BANDS];
  float2* uphist[SPIIR_MAX_BANDS];      // [det][T][kUpHist] for bands above out_band
  const int32_t* tb_first;              // [T][B]
  const int32_t* tb_count;
  const float* taps_int;                // device [32]
  float2* ring; int64_t ring_len, ring_det_stride;
  float2* snr_out; int32_t n_out;
  long long k0;
  PeakRec* peak;                        // [det][T]
  int32_t B, out_band, T;
  int32_t bufA, bufB;                   // capacities in float2 (incl. history prefix)
  int32_t sb_off[SPIIR_MAX_BANDS], sb_n[SPIIR_MAX_BANDS], sb_total;   // staged band sums in shared memory (float2)
};

void launch_prep(const PrepParams& p, int n_det, cudaStream_t st);
int launch_bank_group(int G, int F, int odd, const BankParams& P, const CtaWork* dev_work, int n_cta, int n_det,
                      int smem, cudaStream_t st);
int launch_combine(const CombineParams& p, int n_det, cudaStream_t st);

// peaks.cu
struct PeakParams {
  const PeakRec* peak;                  // [det][T] from k_combine (mode 0)
  const float2* ring; int64_t ring_len, ring_det_stride;
  unsigned long long* key;              // [det][T] scratch (mode 1)
  long long k0; int32_t n;              // last chunk: first absolute index, samples
  int32_t T, D, bank_size;
  float thr2;
  spiir_trigger* trig; int32_t* count;
};
int launch_peaks(const PeakParams& p, int mode, cudaStream_t st);

}  // namespace spiir

struct spiir_bank_host_band {
  int G = 0, F = 0;
  int n_units = 0, n_units_long = 0;         // padded to whole warps, short first
  int n_wu_short = 0, n_wu_long = 0;
  int Hcap = 0, Hs = 0, cap = 0, reps = 0, nmax = 0, rate = 0, nrep = 4, pad = 0, nsubmax = 0;
  int64_t n_filters = 0;
  // workspace offsets (bytes)
  size_t off_coef2 = 0;
  size_t off_coef = 0, off_off = 0, off_state = 0, off_S = 0, off_x[2] = {0, 0}, off_uphist = 0;
  int prev_n = 0;
};

struct spiir_launch_group {
  int G, F, odd;
  std::vector<spiir::CtaWork> work;
  size_t off_work = 0;
  int smem_bytes = 0;
};

struct spiir_bank {
  spiir_bank_desc desc;          // host pointers inside are NOT kept valid; scalars only
  spiir_bank_host_band band[SPIIR_MAX_BANDS];
  std::vector<spiir_launch_group> groups;
  char* ws = nullptr;
  size_t ws_bytes = 0;
  // workspace offsets
  size_t off_tb_first = 0, off_tb_count = 0, off_taps = 0, off_ring = 0, off_peak = 0, off_m1 = 0;
  size_t bytes_state_total = 0, off_state_begin = 0;   // carried-state region to zero on reset
  int parity = 0;
  int64_t k_next = 0;            // absolute output index of the next chunk's first sample
  int last_n_out = 0;            // output samples of the last chunk
  int64_t last_k0 = 0;
  // optional profiling (spiir_bank_timing_*): 4 events per chunk: call begin, k_bank begin/end, call end
  bool timing = false;
  std::vector<cudaEvent_t> ev_pool;
  size_t ev_used = 0, ev_cap = 0;     // events handed out / enabled (4 per chunk), all created by spiir_bank_timing_enable
};
