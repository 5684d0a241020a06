// Host side of the filter bank: layout planning, workspace carve-up, streaming
// state bookkeeping and the C-ABI entry points spiir_bank_* / spiir_filter_chunk.
// (include/spiir.h documents the contract; DESIGN.md §3-§4 the layout.)
#include <algorithm>
#include <cstdarg>
#include <cstdlib>
#include <cstring>
#include <map>
#include <tuple>
#include <numeric>

#include "spiir_internal.cuh"

namespace spiir {

static thread_local std::string g_error;
static thread_local int64_t g_launches = 0;

void set_error(const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_error = buf;
}
void count_launch(int n) { g_launches += n; }


static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int round_up(int x, int a) { return (x + a - 1) / a * a; }

// Host images of the arrays the plan produces (filled only when `fill` is set).
struct PlanImages {
  std::vector<float4> coef[SPIIR_MAX_BANDS];
  std::vector<float2> coef2[SPIIR_MAX_BANDS];    // a b of a two-sample (odd-only) band
  std::vector<int32_t> off[SPIIR_MAX_BANDS];
  std::vector<int32_t> tb_first, tb_count;
};

static int validate(const spiir_bank_desc* d) {
  SPIIR_REQUIRE(d != nullptr, "desc is NULL");
  SPIIR_REQUIRE(d->n_det >= 1 && d->n_det <= SPIIR_MAX_DET, "n_det %d out of range", d->n_det);
  SPIIR_REQUIRE(d->n_templates >= 1, "n_templates %d", d->n_templates);
  SPIIR_REQUIRE(d->n_bands >= 1 && d->n_bands <= SPIIR_MAX_BANDS, "n_bands %d out of range", d->n_bands);
  SPIIR_REQUIRE(d->out_band >= 0 && d->out_band <= 1 && d->out_band < d->n_bands, "out_band %d must be 0 or 1",
                d->out_band);
  for (int b = 0; b + 1 < d->n_bands; ++b)
    SPIIR_REQUIRE(d->band_rate_hz[b] == 2 * d->band_rate_hz[b + 1], "band rates must halve (band %d)", b);
  SPIIR_REQUIRE(d->host_tmpl_offset && d->host_a && d->host_b && d->host_delay && d->host_band,
                "a filter array is NULL");
  SPIIR_REQUIRE(d->n_bands == 1 || (d->host_fir_dec && d->host_fir_int), "FIR taps are NULL");
  const int gran = 4 << (d->n_bands - 1);
  SPIIR_REQUIRE(d->max_chunk_samples >= gran && d->max_chunk_samples % gran == 0,
                "max_chunk_samples %d must be a positive multiple of %d", d->max_chunk_samples, gran);
  SPIIR_REQUIRE(d->n_bands == 1 || d->max_chunk_samples <= 4096, "max_chunk_samples > 4096 with several bands");
  SPIIR_REQUIRE(d->max_chunk_samples <= 8192, "max_chunk_samples > 8192");
  SPIIR_REQUIRE(d->ring_len >= (d->max_chunk_samples >> d->out_band), "ring_len shorter than one chunk");
  SPIIR_REQUIRE(d->host_tmpl_offset[0] == 0 && d->host_tmpl_offset[d->n_templates] == d->n_filters,
                "tmpl_offset does not span n_filters");
  for (int t = 0; t < d->n_templates; ++t)
    SPIIR_REQUIRE(d->host_tmpl_offset[t + 1] >= d->host_tmpl_offset[t], "tmpl_offset not monotone at %d", t);
  for (int b = 0; b < d->n_bands; ++b) SPIIR_REQUIRE(d->max_delay[b] >= 0, "max_delay[%d] < 0", b);
  SPIIR_REQUIRE(d->bank_size >= 1, "bank_size %d must be >= 1", d->bank_size);
  SPIIR_REQUIRE((d->n_templates + d->bank_size - 1) / d->bank_size <= 65535, "too many template banks");
  for (int64_t l = 0; l < d->n_filters; ++l) {
    const int b = d->host_band[l];
    SPIIR_REQUIRE(b >= 0 && b < d->n_bands, "filter %lld: band %d out of range", (long long)l, b);
    SPIIR_REQUIRE(d->host_delay[l] >= 0 && d->host_delay[l] <= d->max_delay[b],
                  "filter %lld: delay %d outside [0, max_delay[%d]=%d]", (long long)l, d->host_delay[l], b,
                  d->max_delay[b]);
  }
  return SPIIR_OK;
}

// Chooses lanes-per-unit G and filters-per-lane F of a band: fewest issue slots
// for the band's templates (8F FP32 per lane-sample + load + reduction share).
static void choose_shape(const std::vector<int>& cnt, int* G_out, int* F_out) {
  double best = 1e300;
  for (int G : {8, 16, 32})
    for (int F = 4; F <= 12; ++F) {
      const double red = (G == 8 ? 28.0 : G == 16 ? 30.0 : 32.0) / 4.0;
      double cost = 0;
      for (int c : cnt)
        if (c > 0) cost += (double)((c + G * F - 1) / (G * F)) * G * (8.0 * F + 0.25 * F + red + 1.0);
      if (cost < best) { best = cost; *G_out = G; *F_out = F; }
    }
}

// Builds the whole device layout.  With img == nullptr only sizes are computed.
static int plan(const spiir_bank_desc* d, spiir_bank* bk, PlanImages* img) {
  const int B = d->n_bands, T = d->n_templates, D = d->n_det;
  bk->desc = *d;
  bk->groups.clear();
  size_t cur = 0;
  auto take = [&](size_t bytes) { size_t o = cur; cur = align_up(cur + bytes, 256); return o; };
  if (img) { img->tb_first.assign((size_t)T * B, 0); img->tb_count.assign((size_t)T * B, 0); }

  // per band: filters of each template
  std::vector<std::vector<int64_t>> ids((size_t)T);
  std::map<std::tuple<int, int, int>, size_t> group_of;
  for (int b = 0; b < B; ++b) {
    spiir_bank_host_band& hb = bk->band[b];
    hb = spiir_bank_host_band();
    hb.rate = d->band_rate_hz[b];
    hb.nmax = d->max_chunk_samples >> b;
    std::vector<int> cnt(T, 0), maxd(T, 0);
    for (int t = 0; t < T; ++t) {
      ids[t].clear();
      for (int64_t l = d->host_tmpl_offset[t]; l < d->host_tmpl_offset[t + 1]; ++l)
        if (d->host_band[l] == b) { ids[t].push_back(l); maxd[t] = std::max(maxd[t], d->host_delay[l]); }
      cnt[t] = (int)ids[t].size();
      hb.n_filters += cnt[t];
    }
    choose_shape(cnt, &hb.G, &hb.F);
    const int G = hb.G, F = hb.F, cap_unit = G * F, upw = 32 / G;
    const int odd = (b == 0 && d->out_band == 1) ? 1 : 0;      // the band above the output rate: two samples per step
    // That band's launch is bound by shared-memory bandwidth, a third of it bank conflicts between the 8 lanes of an
    // LDS.128 phase (profiles/r2_ncu_summary.md section 3): it gets 8 shifted replicas instead of 4, so that every filter
    // has TWO aligned places to read its samples from (replica al or al + 4: a different 16-byte bank group) and the
    // placement below can balance the groups; the staged sub-chunk shrinks to 1024 samples to keep two CTAs per SM.
    hb.nrep = odd ? kReplicas2 : kReplicas;
    hb.pad = odd ? 4 : 0;
    hb.Hcap = std::max(32, round_up(d->max_delay[b], 4)) + hb.pad;
    int nsubmax = std::min(hb.nmax, kSubChunkMax);
    if (hb.nrep == kReplicas2) nsubmax = std::min(nsubmax, 1024);
    hb.nsubmax = nsubmax;
    // shared history depth: the deepest template that still fits the shared-memory budget;
    // templates beyond it (chirp-matched ones) read their input from L1/L2
    {
      const int budget = (kSmemFloatsMax * kReplicas / hb.nrep - nsubmax - hb.pad) / 4 * 4;
      int h = 0;
      for (int t = 0; t < T; ++t) if (cnt[t] && maxd[t] <= budget) h = std::max(h, maxd[t]);
      hb.Hs = std::min(std::max(round_up(h, 4), 4), hb.Hcap - hb.pad);
    }
    hb.cap = round_up(hb.Hcap + hb.nmax + 4, 32);
    hb.reps = hb.pad + hb.Hs + nsubmax;
    // units: short classes first
    std::vector<int> first(T, 0), nun(T, 0);
    int nus = 0, nul = 0;
    for (int t = 0; t < T; ++t) {
      nun[t] = (cnt[t] + cap_unit - 1) / cap_unit;
      if (cnt[t] && maxd[t] <= hb.Hs) { first[t] = nus; nus += nun[t]; }
    }
    const int nus_pad = round_up(nus, upw);
    for (int t = 0; t < T; ++t)
      if (cnt[t] && maxd[t] > hb.Hs) { first[t] = nus_pad + nul; nul += nun[t]; }
    const int nul_pad = round_up(nul, upw);
    hb.n_units = nus_pad + nul_pad;
    hb.n_units_long = nul_pad;
    hb.n_wu_short = nus_pad / upw;
    hb.n_wu_long = nul_pad / upw;
    const size_t slots = (size_t)hb.n_units * cap_unit;
    hb.off_coef = take(slots * sizeof(float4));
    if (odd) hb.off_coef2 = take(slots * sizeof(float2));
    hb.off_off = take(slots * sizeof(int32_t));
    // launch groups, one per (G, F); the long-delay CTAs of a group are listed first (they start first
    // and overlap the rest instead of forming a tail)
    for (int cls = 1; cls >= 0; --cls) {
      const int nwu = cls ? hb.n_wu_long : hb.n_wu_short;
      if (!nwu) continue;
      auto key = std::make_tuple(G, F, odd);
      if (!group_of.count(key)) {
        group_of[key] = bk->groups.size();
        spiir_launch_group g; g.G = G; g.F = F; g.odd = odd;
        bk->groups.push_back(g);
      }
      spiir_launch_group& g = bk->groups[group_of[key]];
      const int wu0 = cls ? hb.n_wu_short : 0;
      std::vector<CtaWork> add;
      for (int w = 0; w < nwu; w += kBankWarps)
        add.push_back(CtaWork{b, wu0 + w, wu0 + std::min(nwu, w + kBankWarps), cls});
      if (cls) g.work.insert(g.work.begin(), add.begin(), add.end());
      else     g.work.insert(g.work.end(), add.begin(), add.end());
      if (!cls) g.smem_bytes = std::max(g.smem_bytes, hb.nrep * hb.reps * 4 + 16);
    }
    if (img) {
      img->coef[b].assign(slots, make_float4(0.f, 0.f, 0.f, 0.f));
      if (odd) img->coef2[b].assign(slots, make_float2(0.f, 0.f));
      img->off[b].assign(slots, 0);
      const int prpu = F * (G / 8);                          // phase-rows per unit
      std::vector<std::pair<int, int64_t>> order;
      std::vector<int> row_fill, row_max, row_cls;
      std::vector<std::pair<int, int>> place;
      for (int t = 0; t < T; ++t) {
        img->tb_first[(size_t)t * B + b] = first[t];
        img->tb_count[(size_t)t * B + b] = nun[t];
        if (!cnt[t]) continue;
        const bool lng = maxd[t] > hb.Hs;
        // where a filter may read its samples: `off` = float offset of its first sample in the staged replica set (or,
        // for the long-delay class, in the global one), and the 16-byte bank group it starts in.  With 8 replicas a
        // filter has two choices (replica al or al + 4).
        const bool two = !lng && hb.nrep == kReplicas2;
        auto choice = [&](int64_t l, int which, int* off_out) {
          const int dl = d->host_delay[l];
          const int e = lng ? hb.Hcap - dl : hb.pad + hb.Hs - dl;
          const int r = (e & 3) + 4 * which;
          const int off = r * (lng ? hb.cap : hb.reps) + (e - r);
          if (off_out) *off_out = off;
          return (off >> 2) & 7;
        };
        order.clear();
        for (int64_t l : ids[t]) order.push_back({choice(l, 0, nullptr), l});
        // Place the filters on the phase-rows (8 lanes x one LDS.128 = one shared-memory wavefront when
        // the 8 addresses fall in 8 different 16-byte bank groups).  A row costs as many wavefronts as its
        // most frequent group, so with one choice per filter the total cannot go below the size of the template's
        // largest group; dealing class by class, largest first, each filter to the row (and, with two replicas to
        // choose from, the replica) where it raises that maximum least, lands the surplus of every oversubscribed
        // group in the same rows (one choice, uniformly random groups: 1.44 wavefronts per row against 1.64 for a plain
        // round-robin, bound 1.42; measured on config 4: bank conflicts of the band-0 launch 4.7e8 -> 3.7e8).
        std::stable_sort(order.begin(), order.end(),
                         [](const std::pair<int, int64_t>& x, const std::pair<int, int64_t>& y) { return x.first < y.first; });
        const int PR = nun[t] * prpu;
        int ccnt[8] = {0, 0, 0, 0, 0, 0, 0, 0}, cbeg[9];
        for (const auto& o : order) ++ccnt[o.first];
        cbeg[0] = 0;
        for (int c = 0; c < 8; ++c) cbeg[c + 1] = cbeg[c] + ccnt[c];
        int corder[8] = {0, 1, 2, 3, 4, 5, 6, 7};
        std::stable_sort(corder, corder + 8, [&](int x, int y) { return ccnt[x] > ccnt[y]; });
        row_fill.assign(PR, 0); row_max.assign(PR, 0); row_cls.assign((size_t)PR * 8, 0);
        place.assign(order.size(), std::pair<int, int>(0, 0));
        std::vector<int> which_of(order.size(), 0);
        if (two) {
          // Two choices per filter: first balance the GROUPS — every filter takes one of its two bank groups so that no
          // group holds more filters than there are rows (PR); then a group's filters go to distinct rows, and a row (8
          // lanes, 8 groups) never sees a group twice: no conflict at all when the balance exists.  The balance is a
          // tiny flow problem (8 groups): start from the less loaded choice, then move filters along augmenting paths
          // from overfull groups to groups with room.
          const int nf = (int)order.size();
          std::vector<int> g0(nf), g1(nf), cur(nf);
          int load[8] = {0, 0, 0, 0, 0, 0, 0, 0};
          for (int j = 0; j < nf; ++j) {
            g0[j] = order[j].first; g1[j] = choice(order[j].second, 1, nullptr);
            which_of[j] = load[g1[j]] < load[g0[j]] ? 1 : 0;
            cur[j] = which_of[j] ? g1[j] : g0[j];
            ++load[cur[j]];
          }
          for (int guard = 0; guard < 8 * nf; ++guard) {
            int over = -1;
            for (int g = 0; g < 8; ++g) if (load[g] > PR && (over < 0 || load[g] > load[over])) over = g;
            if (over < 0) break;
            // breadth-first search over groups from `over` to any group with room, along filters that can switch
            int prev_f[8], seen[8] = {0, 0, 0, 0, 0, 0, 0, 0}, queue[8], qh = 0, qt = 0, target = -1;
            queue[qt++] = over; seen[over] = 1; prev_f[over] = -1;
            while (qh < qt && target < 0) {
              const int g = queue[qh++];
              for (int j = 0; j < nf && target < 0; ++j) {
                if (cur[j] != g) continue;
                const int h = which_of[j] ? g0[j] : g1[j];
                if (seen[h]) continue;
                seen[h] = 1; prev_f[h] = j; queue[qt++] = h;
                if (load[h] < PR) target = h;
              }
            }
            if (target < 0) break;                                    // no balance exists: the surplus stays (conflicts)
            for (int h = target; prev_f[h] >= 0;) {                   // switch the filters on the path, back to front
              const int j = prev_f[h], g = cur[j];
              which_of[j] ^= 1; cur[j] = h; ++load[h]; --load[g];
              h = g;
            }
          }
          // rows: a group's filters to distinct rows, emptiest rows first; a surplus beyond PR wraps around
          for (int g = 0; g < 8; ++g) {
            std::vector<int> rows_by_fill(PR);
            for (int r = 0; r < PR; ++r) rows_by_fill[r] = r;
            std::stable_sort(rows_by_fill.begin(), rows_by_fill.end(), [&](int x, int y) { return row_fill[x] < row_fill[y]; });
            int k = 0;
            for (int j = 0; j < nf; ++j) {
              if (cur[j] != g) continue;
              int r = rows_by_fill[k % PR];
              for (int tries = 0; row_fill[r] >= 8 && tries < PR; ++tries) r = rows_by_fill[(++k) % PR];
              place[j] = std::pair<int, int>(r, row_fill[r]);
              ++row_fill[r];
              ++k;
            }
          }
        } else
        for (int ci = 0; ci < 8; ++ci) {
          const int c0 = corder[ci];
          for (int j = cbeg[c0]; j < cbeg[c0 + 1]; ++j) {
            int best = -1; long best_key = 0;
            for (int r = 0; r < PR; ++r) {
              if (row_fill[r] >= 8) continue;
              const int have = row_cls[(size_t)r * 8 + c0];
              const long key = ((long)std::max(0, have + 1 - row_max[r]) << 40) | ((long)have << 20) | (long)row_fill[r];
              if (best < 0 || key < best_key) { best = r; best_key = key; }
            }
            place[j] = std::pair<int, int>(best, row_fill[best]);
            ++row_fill[best];
            row_max[best] = std::max(row_max[best], ++row_cls[(size_t)best * 8 + c0]);
          }
        }
        for (size_t j = 0; j < order.size(); ++j) {
          const int64_t l = order[j].second;
          const int pr = place[j].first, pos = place[j].second;
          const int ul = pr / prpu, rem = pr % prpu, f = rem / (G / 8), half = rem % (G / 8);
          const int unit = first[t] + ul, g8 = half * 8 + pos;
          const int wu = unit / upw, lane = (unit % upw) * G + g8;
          const size_t slot = ((size_t)wu * F + f) * 32 + lane;
          img->coef[b][slot] = make_float4(d->host_a[l].re, d->host_a[l].im, d->host_b[l].re, d->host_b[l].im);
          if (odd) {                                           // a^2 and a b in float64 from the float32 a, b, rounded once
            const double ar = d->host_a[l].re, ai = d->host_a[l].im, br = d->host_b[l].re, bi = d->host_b[l].im;
            img->coef[b][slot].x = (float)(ar * ar - ai * ai);
            img->coef[b][slot].y = (float)(2.0 * ar * ai);
            img->coef2[b][slot] = make_float2((float)(ar * br - ai * bi), (float)(ar * bi + ai * br));
          }
          int off = 0;
          choice(l, which_of[j], &off);
          img->off[b][slot] = off;
        }
      }
    }
  }
  // carried state (zeroed by reset) is laid out contiguously
  bk->off_state_begin = cur;
  for (int b = 0; b < B; ++b) {
    spiir_bank_host_band& hb = bk->band[b];
    const size_t slots = (size_t)hb.n_units * hb.G * hb.F;
    hb.off_state = take((size_t)D * slots * sizeof(float2));
    hb.off_x[0] = take((size_t)D * hb.nrep * hb.cap * sizeof(float));
    hb.off_x[1] = take((size_t)D * hb.nrep * hb.cap * sizeof(float));
    hb.off_uphist = take((size_t)D * T * kUpHist * sizeof(float2));
  }
  bk->off_peak = take((size_t)D * T * sizeof(PeakRec));
  bk->off_ring = take((size_t)D * T * (size_t)d->ring_len * sizeof(float2));
  bk->bytes_state_total = cur - bk->off_state_begin;
  for (int b = 0; b < B; ++b) {
    spiir_bank_host_band& hb = bk->band[b];
    hb.off_S = take((size_t)D * hb.n_units * hb.nmax * sizeof(float2));
  }
  bk->off_tb_first = take((size_t)T * B * sizeof(int32_t));
  bk->off_tb_count = take((size_t)T * B * sizeof(int32_t));
  bk->off_taps = take(2 * SPIIR_FIR_TAPS * sizeof(float));
  const int n_out_max = d->max_chunk_samples >> d->out_band;
  const int n_banks = (T + std::max(1, d->bank_size) - 1) / std::max(1, d->bank_size);
  (void)n_out_max; (void)n_banks;
  bk->off_m1 = take((size_t)D * T * sizeof(unsigned long long));
  for (auto& g : bk->groups) g.off_work = take(g.work.size() * sizeof(CtaWork));
  bk->ws_bytes = cur;
  return SPIIR_OK;
}

}  // namespace spiir

using namespace spiir;

extern "C" {

const char* spiir_last_error(void) { return g_error.c_str(); }
int64_t spiir_launch_count(void) { return g_launches; }

int spiir_bank_workspace_bytes(const spiir_bank_desc* desc, size_t* bytes) {
  int rc = validate(desc);
  if (rc) return rc;
  SPIIR_REQUIRE(bytes != nullptr, "bytes is NULL");
  spiir_bank tmp;
  rc = plan(desc, &tmp, nullptr);
  if (rc) return rc;
  *bytes = tmp.ws_bytes;
  return SPIIR_OK;
}

int spiir_bank_init(spiir_bank** out, const spiir_bank_desc* desc, void* dev_workspace, size_t bytes, void* stream) {
  int rc = validate(desc);
  if (rc) return rc;
  SPIIR_REQUIRE(out && dev_workspace, "out or workspace is NULL");
  SPIIR_REQUIRE(((uintptr_t)dev_workspace & 255) == 0, "workspace must be 256-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  spiir_bank* bk = new spiir_bank();
  PlanImages img;
  rc = plan(desc, bk, &img);
  if (rc) { delete bk; return rc; }
  if (bytes < bk->ws_bytes) {
    set_error("workspace too small: %zu < %zu", bytes, bk->ws_bytes);
    delete bk;
    return SPIIR_ENOMEM;
  }
  bk->ws = (char*)dev_workspace;
  auto fail = [&](cudaError_t e, const char* what) {
    set_error("%s failed: %s", what, cudaGetErrorString(e));
    delete bk;
    return SPIIR_ECUDA;
  };
  cudaError_t e;
  for (int b = 0; b < desc->n_bands; ++b) {
    auto& hb = bk->band[b];
    if (!img.coef[b].empty()) {
      e = cudaMemcpyAsync(bk->ws + hb.off_coef, img.coef[b].data(), img.coef[b].size() * sizeof(float4),
                          cudaMemcpyHostToDevice, st);
      if (e != cudaSuccess) return fail(e, "copy coef");
      e = cudaMemcpyAsync(bk->ws + hb.off_off, img.off[b].data(), img.off[b].size() * sizeof(int32_t),
                          cudaMemcpyHostToDevice, st);
      if (e != cudaSuccess) return fail(e, "copy off");
      if (!img.coef2[b].empty()) {
        e = cudaMemcpyAsync(bk->ws + hb.off_coef2, img.coef2[b].data(), img.coef2[b].size() * sizeof(float2),
                            cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return fail(e, "copy coef2");
      }
    }
  }
  e = cudaMemcpyAsync(bk->ws + bk->off_tb_first, img.tb_first.data(), img.tb_first.size() * 4, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(e, "copy tb_first");
  e = cudaMemcpyAsync(bk->ws + bk->off_tb_count, img.tb_count.data(), img.tb_count.size() * 4, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(e, "copy tb_count");
  float taps[2 * SPIIR_FIR_TAPS] = {0};
  if (desc->host_fir_dec) memcpy(taps, desc->host_fir_dec, SPIIR_FIR_TAPS * sizeof(float));
  if (desc->host_fir_int) memcpy(taps + SPIIR_FIR_TAPS, desc->host_fir_int, SPIIR_FIR_TAPS * sizeof(float));
  e = cudaMemcpyAsync(bk->ws + bk->off_taps, taps, sizeof(taps), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(e, "copy taps");
  for (auto& g : bk->groups) {
    e = cudaMemcpyAsync(bk->ws + g.off_work, g.work.data(), g.work.size() * sizeof(CtaWork), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return fail(e, "copy work");
  }
  // the host images die with this scope: wait for the copies
  e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail(e, "cudaStreamSynchronize");
  // host pointers of the caller are not kept
  bk->desc.host_tmpl_offset = nullptr; bk->desc.host_a = nullptr; bk->desc.host_b = nullptr;
  bk->desc.host_delay = nullptr; bk->desc.host_band = nullptr; bk->desc.host_fir_dec = nullptr;
  bk->desc.host_fir_int = nullptr;
  rc = spiir_bank_reset(bk, stream);
  if (rc) { delete bk; return rc; }
  *out = bk;
  return SPIIR_OK;
}

int spiir_bank_reset(spiir_bank* bk, void* stream) {
  SPIIR_REQUIRE(bk != nullptr, "bank is NULL");
  SPIIR_CUDA_OK(cudaMemsetAsync(bk->ws + bk->off_state_begin, 0, bk->bytes_state_total, (cudaStream_t)stream));
  bk->parity = 0;
  bk->k_next = 0;
  bk->last_n_out = 0;
  bk->last_k0 = 0;
  for (int b = 0; b < bk->desc.n_bands; ++b) bk->band[b].prev_n = 0;
  return SPIIR_OK;
}

int spiir_bank_timing_enable(spiir_bank* bk, int32_t enable) {
  SPIIR_REQUIRE(bk != nullptr, "bank is NULL");
  SPIIR_REQUIRE(enable >= 0 && enable <= (1 << 20), "n_chunks %d out of range", enable);
  // all events are created HERE, so that spiir_filter_chunk itself never creates anything (spiir.h: no allocation
  // after init on the hot path): four per chunk to be recorded
  while (bk->ev_pool.size() < (size_t)enable * 4) {
    cudaEvent_t e;
    SPIIR_CUDA_OK(cudaEventCreate(&e));
    bk->ev_pool.push_back(e);
  }
  bk->timing = enable != 0;
  bk->ev_cap = (size_t)enable * 4;
  bk->ev_used = 0;
  return SPIIR_OK;
}

int spiir_bank_timing_read(spiir_bank* bk, double* ms_recursion, double* ms_chunk, int32_t* n_chunks) {
  SPIIR_REQUIRE(bk && ms_recursion && ms_chunk && n_chunks, "a pointer is NULL");
  double a = 0, c = 0;
  for (size_t i = 0; i + 3 < bk->ev_used; i += 4) {
    float m1 = 0.f, m2 = 0.f;
    SPIIR_CUDA_OK(cudaEventSynchronize(bk->ev_pool[i + 3]));
    SPIIR_CUDA_OK(cudaEventElapsedTime(&m1, bk->ev_pool[i + 1], bk->ev_pool[i + 2]));
    SPIIR_CUDA_OK(cudaEventElapsedTime(&m2, bk->ev_pool[i], bk->ev_pool[i + 3]));
    a += m1; c += m2;
  }
  *ms_recursion = a; *ms_chunk = c; *n_chunks = (int32_t)(bk->ev_used / 4);
  bk->ev_used = 0;
  return SPIIR_OK;
}

int spiir_bank_free(spiir_bank* bk) {
  SPIIR_REQUIRE(bk != nullptr, "bank is NULL");
  for (cudaEvent_t e : bk->ev_pool) cudaEventDestroy(e);
  delete bk;
  return SPIIR_OK;
}

int spiir_filter_chunk(spiir_bank* bk, const float* dev_strain, int32_t n_samples, spiir_c32* dev_snr_out,
                       void* stream) {
  SPIIR_REQUIRE(bk != nullptr && dev_strain != nullptr, "bank or strain is NULL");
  const spiir_bank_desc& d = bk->desc;
  const int B = d.n_bands, D = d.n_det, T = d.n_templates;
  const int gran = 4 << (B - 1);
  SPIIR_REQUIRE(n_samples > 0 && n_samples % gran == 0 && n_samples <= d.max_chunk_samples,
                "n_samples %d must be a positive multiple of %d and <= %d", n_samples, gran, d.max_chunk_samples);
  SPIIR_REQUIRE(((uintptr_t)dev_strain & 15) == 0, "dev_strain must be 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  const int newp = bk->parity ^ 1;

  PrepParams pp;
  memset(&pp, 0, sizeof(pp));
  pp.strain = dev_strain; pp.n0 = n_samples; pp.n_bands = B;
  pp.taps_dec = (const float*)(bk->ws + bk->off_taps);
  BankParams P;
  memset(&P, 0, sizeof(P));
  for (int b = 0; b < B; ++b) {
    auto& hb = bk->band[b];
    const int n = n_samples >> b;
    pp.xnew[b] = (float*)(bk->ws + hb.off_x[newp]);
    pp.xold[b] = (const float*)(bk->ws + hb.off_x[bk->parity]);
    pp.x_det_stride[b] = (int64_t)hb.nrep * hb.cap;
    pp.nrep[b] = hb.nrep;
    pp.cap[b] = hb.cap; pp.Hcap[b] = hb.Hcap; pp.n[b] = n; pp.prev_n[b] = hb.prev_n;
    BandDev& bd = P.band[b];
    const size_t slots = (size_t)hb.n_units * hb.G * hb.F;
    bd.coef = (const float4*)(bk->ws + hb.off_coef);
    bd.coef2 = (const float2*)(bk->ws + hb.off_coef2);
    bd.off = (const int32_t*)(bk->ws + hb.off_off);
    bd.state = (float2*)(bk->ws + hb.off_state);
    bd.S = (float2*)(bk->ws + hb.off_S);
    bd.xrep = pp.xnew[b];
    bd.x_det_stride = pp.x_det_stride[b];
    bd.state_det_stride = (int64_t)slots;
    bd.S_det_stride = (int64_t)hb.n_units * hb.nmax;
    bd.n = n; bd.nmax = hb.nmax; bd.Hcap = hb.Hcap; bd.Hs = hb.Hs; bd.cap = hb.cap; bd.reps = hb.reps;
    bd.nsub = std::min(n, hb.nsubmax);
    bd.nrep = hb.nrep; bd.pad = hb.pad;
    bd.odd = (b == 0 && d.out_band == 1) ? 1 : 0;
  }
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  const bool timed = bk->timing && bk->ev_used + 4 <= bk->ev_cap;     // chunks beyond the enabled count go unrecorded
  if (timed) {
    for (int i = 0; i < 4; ++i) ev[i] = bk->ev_pool[bk->ev_used + i];
    bk->ev_used += 4;
    SPIIR_CUDA_OK(cudaEventRecord(ev[0], st));
  }
  launch_prep(pp, D, st);
  SPIIR_CUDA_OK(cudaGetLastError());
  if (timed) SPIIR_CUDA_OK(cudaEventRecord(ev[1], st));
  for (auto& g : bk->groups) {
    int rc = launch_bank_group(g.G, g.F, g.odd, P, (const CtaWork*)(bk->ws + g.off_work), (int)g.work.size(), D,
                               g.smem_bytes, st);
    if (rc) return rc;
  }
  if (timed) SPIIR_CUDA_OK(cudaEventRecord(ev[2], st));
  CombineParams cp;
  memset(&cp, 0, sizeof(cp));
  for (int b = 0; b < B; ++b) {
    auto& hb = bk->band[b];
    cp.S[b] = (const float2*)(bk->ws + hb.off_S);
    cp.S_det_stride[b] = (int64_t)hb.n_units * hb.nmax;
    cp.nmax[b] = hb.nmax; cp.n[b] = n_samples >> b;
    cp.uphist[b] = (float2*)(bk->ws + hb.off_uphist);
  }
  cp.tb_first = (const int32_t*)(bk->ws + bk->off_tb_first);
  cp.tb_count = (const int32_t*)(bk->ws + bk->off_tb_count);
  cp.taps_int = (const float*)(bk->ws + bk->off_taps) + SPIIR_FIR_TAPS;
  cp.ring = (float2*)(bk->ws + bk->off_ring);
  cp.ring_len = d.ring_len; cp.ring_det_stride = (int64_t)T * d.ring_len;
  cp.snr_out = (float2*)dev_snr_out;
  cp.n_out = n_samples >> d.out_band;
  cp.k0 = bk->k_next;
  cp.peak = (PeakRec*)(bk->ws + bk->off_peak);
  cp.B = B; cp.out_band = d.out_band; cp.T = T;
  cp.bufA = (kUpHist + (d.max_chunk_samples >> d.out_band) + 4) & ~1;   // even, and room for the 17-sample window reads
  cp.bufB = (B - 1 > d.out_band) ? (kUpHist + (d.max_chunk_samples >> (d.out_band + 1)) + 4) & ~1 : 0;
  cp.sb_total = 0;
  for (int b = 0; b < B; ++b) {
    const int n = n_samples >> b;
    cp.sb_n[b] = (b == 0 && d.out_band == 1) ? n / 2 : n;
    cp.sb_off[b] = cp.sb_total;
    cp.sb_total += (cp.sb_n[b] + 1) & ~1;
  }
  { const int rcc = launch_combine(cp, D, st); if (rcc) return rcc; }
  if (timed) SPIIR_CUDA_OK(cudaEventRecord(ev[3], st));

  bk->parity = newp;
  for (int b = 0; b < B; ++b) bk->band[b].prev_n = n_samples >> b;
  bk->last_k0 = bk->k_next;
  bk->last_n_out = cp.n_out;
  bk->k_next += cp.n_out;
  return SPIIR_OK;
}

int spiir_peaks(spiir_bank* bk, float snr_threshold, int32_t mode, spiir_trigger* dev_trig, int32_t* dev_count,
                void* stream) {
  SPIIR_REQUIRE(bk && dev_trig && dev_count, "bank, dev_trig or dev_count is NULL");
  SPIIR_REQUIRE(mode == 0 || mode == 1, "mode %d must be 0 or 1", mode);
  SPIIR_REQUIRE(snr_threshold >= 0.f, "snr_threshold must be >= 0");
  SPIIR_REQUIRE(bk->last_n_out > 0, "spiir_peaks before the first spiir_filter_chunk");
  const spiir_bank_desc& d = bk->desc;
  PeakParams p;
  memset(&p, 0, sizeof(p));
  p.peak = (const PeakRec*)(bk->ws + bk->off_peak);
  p.ring = (const float2*)(bk->ws + bk->off_ring);
  p.ring_len = d.ring_len; p.ring_det_stride = (int64_t)d.n_templates * d.ring_len;
  p.key = (unsigned long long*)(bk->ws + bk->off_m1);
  p.k0 = bk->last_k0; p.n = bk->last_n_out;
  p.T = d.n_templates; p.D = d.n_det; p.bank_size = d.bank_size;
  p.thr2 = snr_threshold * snr_threshold;       // float32 product, as the oracle's decision path
  p.trig = dev_trig; p.count = dev_count;
  return launch_peaks(p, mode, (cudaStream_t)stream);
}

int spiir_bank_snr_view(const spiir_bank* bk, spiir_snr_view* view) {
  SPIIR_REQUIRE(bk && view, "bank or view is NULL");
  view->dev_z = (const spiir_c32*)(bk->ws + bk->off_ring);
  view->row_stride = bk->desc.ring_len;
  view->det_stride = (int64_t)bk->desc.n_templates * bk->desc.ring_len;
  view->ring_len = bk->desc.ring_len;
  view->k_newest = bk->k_next - 1;
  view->n_rows = bk->desc.n_templates;
  return SPIIR_OK;
}

int spiir_bank_band_plan(const spiir_bank* bk, int32_t band, spiir_band_plan* p) {
  SPIIR_REQUIRE(bk && p && band >= 0 && band < bk->desc.n_bands, "bad arguments");
  const auto& hb = bk->band[band];
  p->lanes_per_unit = hb.G; p->filters_per_lane = hb.F;
  p->n_units = hb.n_units; p->n_units_long = hb.n_units_long;
  p->smem_history = hb.Hs; p->smem_bytes = hb.nrep * hb.reps * 4 + 16;
  p->n_filters = hb.n_filters; p->n_slots = (int64_t)hb.n_units * hb.G * hb.F;
  return SPIIR_OK;
}

int64_t spiir_bank_updates_per_chunk(const spiir_bank* bk, int32_t n_samples) {
  if (!bk) return 0;
  int64_t u = 0;
  for (int b = 0; b < bk->desc.n_bands; ++b) u += bk->band[b].n_filters * (int64_t)(n_samples >> b);
  return u * bk->desc.n_det;
}

}  // extern "C"
