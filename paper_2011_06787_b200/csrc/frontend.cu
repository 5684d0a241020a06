// NEXT-4 — the front end of the pipeline on the device (Sec. II A; latencies PAPER.md:354):
//   FIR down-sampling (16 384 -> 2048 Hz, N_FIR ~ 192)  ->  frequency-domain whitening, Eq. 1, against the running
//   median PSD of the immediate past (overlapping 4-s blocks spanning 56 s)  ->  amplitude gating with 0.25 s of
//   zeros on either side.  Readings W1-W6: DESIGN.md section 11d (the oracle is oracle/frontend.py).
//
// One call consumes one hop of H output samples per detector (2 s at 2048 Hz) and emits the H gated samples whose
// whitening that hop completes.  Work per call is tiny (3 detectors x one 8192-point transform), so the whole
// stage is ONE kernel, one CTA of 1024 threads per detector, everything between the raw samples and the output
// in shared memory: FIR -> Hann window -> radix-2 FFT (decimation in frequency, natural in / bit-reversed out) ->
// periodogram into the history ring, median over the past blocks per frequency bin -> division in bit-reversed
// order -> inverse FFT (decimation in time, bit-reversed in / natural out: no re-ordering pass anywhere) ->
// overlap-add -> gate.  The transform is hand-written (no cuFFT on the path); twiddles and the window are formed in
// float64 on the host.  It is latency-bound by its 2 x log2(2H) barrier-separated stages; bench.py reports its time.
#include <cmath>
#include <cstring>
#include <vector>

#include "spiir_internal.cuh"

namespace spiir {

constexpr int kFeThreads = 1024;
constexpr int kFeMaxHist = 31;

struct FeParams {
  const float* raw; float* out; float* psd_out;      // [n_det][H R], [n_det][H], [n_det][H + 1] or null
  const float* taps; const float2* tw; const float* win; const float* inv_bias;   // [n_taps], [N/2], [N], [n_hist + 1]
  float* raw_hist; float* prev_hop; float* tail; float* carry; float* P;           // carried state, per detector
  int32_t H, N, logN, R, n_taps, n_hist, pad;
  int32_t call;                                       // index c of this call since the last reset
  float p_norm;                                       // 2 / (f_s sum w^2)
  float half_fs;                                      // f_s / 2
  float thr;
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

__global__ void __launch_bounds__(kFeThreads, 1) k_frontend(const __grid_constant__ FeParams P) {
  extern __shared__ __align__(16) unsigned char fe_smem[];
  const int H = P.H, N = P.N, tid = threadIdx.x, det = blockIdx.x;
  float2* X = reinterpret_cast<float2*>(fe_smem);                 // [N] the block, time or frequency domain
  float2* tw = X + N;                                             // [N/2] exp(-2 pi i m / N)
  float* sinv = reinterpret_cast<float*>(tw + N / 2);             // [H + 1] 1 / sqrt(S_n f_s / 2)
  float* taps = sinv + (H + 1);                                   // [n_taps]
  unsigned char* mask = reinterpret_cast<unsigned char*>(taps + P.n_taps);   // [H + 2 pad]
  for (int i = tid; i < N / 2; i += kFeThreads) tw[i] = P.tw[i];
  for (int i = tid; i < P.n_taps; i += kFeThreads) taps[i] = P.taps[i];
  __syncthreads();

  // ---- W1: y[m] = sum_j h[j] x[R m + R - 1 - j]; the n_taps samples before this hop come from the carried history
  const float* raw = P.raw + (size_t)det * H * P.R;
  float* hist = P.raw_hist + (size_t)det * P.n_taps;
  float* prev = P.prev_hop + (size_t)det * H;
  for (int m = tid; m < H; m += kFeThreads) {
    float acc = 0.f;
    const int top = P.R * m + P.R - 1;
    for (int j = 0; j < P.n_taps; ++j) {
      const int i = top - j;
      const float x = i >= 0 ? __ldg(raw + i) : hist[P.n_taps + i];
      acc = fmaf(taps[j], x, acc);
    }
    // block = [hop c-1 | hop c], Hann-windowed (W2)
    X[H + m] = make_float2(acc * __ldg(P.win + H + m), 0.f);
    X[m] = make_float2(prev[m] * __ldg(P.win + m), 0.f);
    prev[m] = acc;                                                 // each thread reads and writes its own elements only
  }
  __syncthreads();
  for (int i = tid; i < P.n_taps; i += kFeThreads) {               // the last n_taps raw samples, for the next call
    const int src = H * P.R - P.n_taps + i;
    hist[i] = src >= 0 ? raw[src] : hist[src + P.n_taps];
  }

  // ---- forward FFT, decimation in frequency: natural order in, bit-reversed order out
  for (int half = N >> 1; half >= 1; half >>= 1) {
    const int tstep = (N >> 1) / half;
    for (int j = tid; j < N / 2; j += kFeThreads) {
      const int pos = j & (half - 1), i = ((j - pos) << 1) + pos;
      const float2 a = X[i], b = X[i + half];
      X[i] = make_float2(a.x + b.x, a.y + b.y);
      X[i + half] = cmul(make_float2(a.x - b.x, a.y - b.y), tw[pos * tstep]);
    }
    __syncthreads();
  }
  // ---- W4: periodogram of this block into the history ring; PSD of the PAST blocks: median per bin / bias
  float* Pd = P.P + (size_t)det * P.n_hist * (H + 1);
  int n = min(P.call, P.n_hist);
  if ((n & 1) == 0) n -= 1;
  const int shift = 32 - P.logN;
  for (int k = tid; k <= H; k += kFeThreads) {
    const float2 d = X[__brev((unsigned)k) >> shift];
    const float pk = P.p_norm * fmaf(d.x, d.x, d.y * d.y);
    float s = 0.f;
    if (n >= 1) {
      float v[kFeMaxHist];
      for (int b = 0; b < n; ++b) {                                 // the n most recent past blocks, insertion-sorted
        const float x = Pd[(size_t)((P.call - 1 - b) % P.n_hist) * (H + 1) + k];
        int q = b;
        while (q > 0 && v[q - 1] > x) { v[q] = v[q - 1]; --q; }
        v[q] = x;
      }
      s = v[n >> 1] * P.inv_bias[n];
    }
    sinv[k] = s > 0.f ? rsqrtf(s * P.half_fs) : 0.f;
    if (P.psd_out) P.psd_out[(size_t)det * (H + 1) + k] = s;
    Pd[(size_t)(P.call % P.n_hist) * (H + 1) + k] = pk;             // read above only for past blocks: distinct slot unless
  }                                                                 // n_hist blocks are in use, and then it is the oldest, read before
  __syncthreads();
  // ---- W3: D_w = D / sqrt(S_n f_s / 2), in bit-reversed order (the frequency of position p is bitrev(p))
  for (int p = tid; p < N; p += kFeThreads) {
    const int k = (int)(__brev((unsigned)p) >> shift);
    const float g = sinv[k <= H ? k : N - k];
    X[p].x *= g; X[p].y *= g;
  }
  __syncthreads();
  // ---- inverse FFT, decimation in time: bit-reversed order in, natural order out
  for (int half = 1; half < N; half <<= 1) {
    const int tstep = (N >> 1) / half;
    for (int j = tid; j < N / 2; j += kFeThreads) {
      const int pos = j & (half - 1), i = ((j - pos) << 1) + pos;
      const float2 w = tw[pos * tstep];
      const float2 a = X[i], t = cmul(X[i + half], make_float2(w.x, -w.y));
      X[i] = make_float2(a.x + t.x, a.y + t.y);
      X[i + half] = make_float2(a.x - t.x, a.y - t.y);
    }
    __syncthreads();
  }
  // ---- overlap-add: hop c-1 is complete; then the gate (W5) on [carry of 2 pad | hop c-1], emitting hop c-1 shifted
  //      by the look-ahead of pad samples (W6)
  float* tail = P.tail + (size_t)det * H;
  float* carry = P.carry + (size_t)det * 2 * P.pad;
  float* dw = reinterpret_cast<float*>(X) + 2 * N - (H + 2 * P.pad);   // upper part of the (now free) transform buffer ...
  const float invN = 1.f / (float)N;
  float keep[8];                                                       // ... whose lower part still holds the block: read first
  for (int u = tid, q = 0; u < H; u += kFeThreads, ++q) {
    keep[q] = tail[u] + X[u].x * invN;
    tail[u] = X[H + u].x * invN;
  }
  __syncthreads();
  for (int u = tid, q = 0; u < H; u += kFeThreads, ++q) dw[2 * P.pad + u] = keep[q];
  for (int u = tid; u < 2 * P.pad; u += kFeThreads) dw[u] = carry[u];
  for (int u = tid; u < H + 2 * P.pad; u += kFeThreads) mask[u] = 0;
  __syncthreads();
  for (int u = tid; u < H + 2 * P.pad; u += kFeThreads) {
    if (fabsf(dw[u]) > P.thr) {
      const int lo = max(0, u - P.pad), hi = min(H + 2 * P.pad - 1, u + P.pad);
      for (int v = lo; v <= hi; ++v) mask[v] = 1;
    }
  }
  __syncthreads();
  float* out = P.out + (size_t)det * H;
  for (int u = tid; u < H; u += kFeThreads) out[u] = mask[P.pad + u] ? 0.f : dw[P.pad + u];
  for (int u = tid; u < 2 * P.pad; u += kFeThreads) carry[u] = dw[H + u];
}

}  // namespace spiir

using namespace spiir;

struct spiir_frontend {
  spiir_frontend_desc d;
  char* ws = nullptr;
  size_t off_taps = 0, off_tw = 0, off_win = 0, off_bias = 0, off_state = 0, state_bytes = 0;
  size_t off_hist = 0, off_prev = 0, off_tail = 0, off_carry = 0, off_P = 0, bytes = 0;
  int N = 0, logN = 0, call = 0;
  double sw2 = 0;
  size_t smem = 0;
};

static int fe_validate(const spiir_frontend_desc* d) {
  SPIIR_REQUIRE(d != nullptr, "desc is NULL");
  SPIIR_REQUIRE(d->n_det >= 1 && d->n_det <= SPIIR_MAX_DET, "n_det %d out of range", d->n_det);
  SPIIR_REQUIRE(d->hop >= 256 && d->hop <= 4096 && (d->hop & (d->hop - 1)) == 0, "hop %d must be a power of two in 256..4096", d->hop);
  SPIIR_REQUIRE(d->decim >= 1 && d->decim <= 16, "decim %d out of range 1..16", d->decim);
  SPIIR_REQUIRE(d->n_taps >= 1 && d->n_taps <= 512 && d->host_taps, "n_taps %d out of range 1..512 or taps NULL", d->n_taps);
  SPIIR_REQUIRE(d->n_taps <= d->hop * d->decim, "n_taps %d longer than one hop of input", d->n_taps);
  SPIIR_REQUIRE(d->n_hist >= 1 && d->n_hist <= kFeMaxHist, "n_hist %d out of range 1..%d", d->n_hist, kFeMaxHist);
  SPIIR_REQUIRE(d->gate_pad >= 0 && 2 * d->gate_pad <= d->hop, "gate_pad %d must be in 0..hop/2", d->gate_pad);
  SPIIR_REQUIRE(d->out_rate_hz > 0.f && d->gate_threshold > 0.f, "out_rate_hz and gate_threshold must be positive");
  return SPIIR_OK;
}

static void fe_layout(spiir_frontend* fe) {
  const spiir_frontend_desc& d = fe->d;
  const int H = d.hop;
  fe->N = 2 * H;
  fe->logN = 0;
  while ((1 << fe->logN) < fe->N) ++fe->logN;
  size_t cur = 0;
  auto take = [&](size_t b) { size_t o = cur; cur = (cur + b + 255) / 256 * 256; return o; };
  fe->off_taps = take((size_t)d.n_taps * 4);
  fe->off_tw = take((size_t)fe->N / 2 * 8);
  fe->off_win = take((size_t)fe->N * 4);
  fe->off_bias = take((size_t)(kFeMaxHist + 1) * 4);
  fe->off_state = cur;
  fe->off_hist = take((size_t)d.n_det * d.n_taps * 4);
  fe->off_prev = take((size_t)d.n_det * H * 4);
  fe->off_tail = take((size_t)d.n_det * H * 4);
  fe->off_carry = take((size_t)d.n_det * (2 * d.gate_pad + 1) * 4);
  fe->off_P = take((size_t)d.n_det * d.n_hist * (H + 1) * 4);
  fe->state_bytes = cur - fe->off_state;
  fe->bytes = cur;
  fe->smem = (size_t)fe->N * 8 + (size_t)fe->N / 2 * 8 + (size_t)(H + 1) * 4 + (size_t)d.n_taps * 4 + (size_t)(H + 2 * d.gate_pad) + 16;
}

// fe_layout's shared-memory formula at the largest shape fe_validate lets through (hop 4096 -> N 8192, 512 taps,
// gate_pad hop / 2): 124 948 bytes, inside the 227 KB a CTA may opt in to.
constexpr size_t kFeSmemMax = (size_t)8192 * 8 + (size_t)4096 * 8 + (size_t)(4096 + 1) * 4 + (size_t)512 * 4 +
                              (size_t)(4096 + 2 * 2048) + 16;

extern "C" {

int spiir_frontend_workspace_bytes(const spiir_frontend_desc* desc, size_t* bytes) {
  int rc = fe_validate(desc);
  if (rc) return rc;
  SPIIR_REQUIRE(bytes != nullptr, "bytes is NULL");
  spiir_frontend fe; fe.d = *desc;
  fe_layout(&fe);
  *bytes = fe.bytes;
  return SPIIR_OK;
}

int spiir_frontend_init(spiir_frontend** out, const spiir_frontend_desc* desc, void* dev_workspace, size_t bytes, void* stream) {
  int rc = fe_validate(desc);
  if (rc) return rc;
  SPIIR_REQUIRE(out && dev_workspace, "out or workspace is NULL");
  SPIIR_REQUIRE(((uintptr_t)dev_workspace & 255) == 0, "workspace must be 256-byte aligned");
  spiir_frontend* fe = new spiir_frontend();
  fe->d = *desc;
  fe_layout(fe);
  if (bytes < fe->bytes) { set_error("workspace too small: %zu < %zu", bytes, fe->bytes); delete fe; return SPIIR_ENOMEM; }
  fe->ws = (char*)dev_workspace;
  const int N = fe->N;
  std::vector<float> tw((size_t)N), win((size_t)N), bias(kFeMaxHist + 1, 0.f);
  const double pi = 3.14159265358979323846;
  for (int m = 0; m < N / 2; ++m) { tw[2 * m] = (float)cos(-2.0 * pi * m / N); tw[2 * m + 1] = (float)sin(-2.0 * pi * m / N); }
  fe->sw2 = 0;
  for (int i = 0; i < N; ++i) { const double w = sin(pi * i / N); win[i] = (float)(w * w); fe->sw2 += w * w * w * w; }
  for (int n = 1; n <= kFeMaxHist; ++n) {               // 1 / bias of the median of n exponential variates (W4)
    double b = 0;
    for (int i = 1; i <= n; ++i) b += ((i & 1) ? 1.0 : -1.0) / i;
    bias[n] = (float)(1.0 / b);
  }
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemcpyAsync(fe->ws + fe->off_taps, desc->host_taps, (size_t)desc->n_taps * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(fe->ws + fe->off_tw, tw.data(), (size_t)N / 2 * 8, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(fe->ws + fe->off_win, win.data(), (size_t)N * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(fe->ws + fe->off_bias, bias.data(), bias.size() * 4, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);       // the host images die with this scope
  if (e != cudaSuccess) { set_error("front-end set-up failed: %s", cudaGetErrorString(e)); delete fe; return SPIIR_ECUDA; }
  fe->d.host_taps = nullptr;
  rc = spiir_frontend_reset(fe, stream);
  if (rc) { delete fe; return rc; }
  *out = fe;
  return SPIIR_OK;
}

int spiir_frontend_reset(spiir_frontend* fe, void* stream) {
  SPIIR_REQUIRE(fe != nullptr, "front end is NULL");
  SPIIR_CUDA_OK(cudaMemsetAsync(fe->ws + fe->off_state, 0, fe->state_bytes, (cudaStream_t)stream));
  fe->call = 0;
  return SPIIR_OK;
}

int spiir_frontend_free(spiir_frontend* fe) {
  SPIIR_REQUIRE(fe != nullptr, "front end is NULL");
  delete fe;
  return SPIIR_OK;
}

int spiir_frontend_chunk(spiir_frontend* fe, const float* dev_raw, float* dev_out, float* dev_psd, void* stream) {
  SPIIR_REQUIRE(fe && dev_raw && dev_out, "front end, dev_raw or dev_out is NULL");
  const spiir_frontend_desc& d = fe->d;
  FeParams P;
  memset(&P, 0, sizeof(P));
  P.raw = dev_raw; P.out = dev_out; P.psd_out = dev_psd;
  P.taps = (const float*)(fe->ws + fe->off_taps); P.tw = (const float2*)(fe->ws + fe->off_tw);
  P.win = (const float*)(fe->ws + fe->off_win); P.inv_bias = (const float*)(fe->ws + fe->off_bias);
  P.raw_hist = (float*)(fe->ws + fe->off_hist); P.prev_hop = (float*)(fe->ws + fe->off_prev);
  P.tail = (float*)(fe->ws + fe->off_tail); P.carry = (float*)(fe->ws + fe->off_carry); P.P = (float*)(fe->ws + fe->off_P);
  P.H = d.hop; P.N = fe->N; P.logN = fe->logN; P.R = d.decim; P.n_taps = d.n_taps; P.n_hist = d.n_hist; P.pad = d.gate_pad;
  P.call = fe->call;
  P.p_norm = (float)(2.0 / ((double)d.out_rate_hz * fe->sw2));
  P.half_fs = 0.5f * d.out_rate_hz;
  P.thr = d.gate_threshold;
  // The opt-in shared-memory limit is a property of the FUNCTION on a device, not of this instance: it is set once
  // per device, to what the largest valid descriptor needs, so that instances of different shapes never lower it
  // for one another and a front end works on whichever device is current when it is run.
  static unsigned long long configured = 0;
  if (first_use_on_device(configured))
    SPIIR_CUDA_OK(cudaFuncSetAttribute(k_frontend, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFeSmemMax));
  SPIIR_REQUIRE(fe->smem <= kFeSmemMax, "front end needs %zu bytes of shared memory (> %zu)", fe->smem, kFeSmemMax);
  k_frontend<<<d.n_det, kFeThreads, fe->smem, (cudaStream_t)stream>>>(P);
  count_launch();
  SPIIR_CUDA_OK(cudaGetLastError());
  fe->call += 1;
  return SPIIR_OK;
}

}  // extern "C"
