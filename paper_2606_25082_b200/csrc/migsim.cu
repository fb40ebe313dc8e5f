// migsim.cu -- host side of libmigsim.so: the C ABI of include/migsim.h (argument checking, table preparation, launches).
// Every step of the simulated path runs in the kernels of sim_device.cuh / qnet_device.cuh; there is no CPU fallback.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>
#include <vector>

#include "qnet_device.cuh"
#include "sim_device.cuh"
#include "sim_thread.cuh"

using namespace migsim;

// ------------------------------------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
static int fail(int code, const char *fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap);
  return code;
}
// the same for the other translation units of the library (dqn.cu)
int mig_fail(int code, const char *fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof(g_err), fmt, ap); va_end(ap);
  return code;
}
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(MIG_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); } while (0)

extern "C" const char *mig_last_error(void) { return g_err; }
extern "C" const char *mig_version(void) { return "migsim 0.1 sm_100a (" __DATE__ ")"; }

// ------------------------------------------------------------------------------------------------ handles
struct mig_qnet {
  float *d = nullptr;        // one allocation: W1 b1 W2 b2 W3 b3
  const float *W1, *b1, *W2, *b2, *W3, *b3;
  uint32_t H = 0, A = 0;
  int device = 0;
};

struct mig_sim {
  mig_params_t p;            // scalars (pointers inside are NOT kept)
  uint32_t n_envs = 0; uint64_t seed = 0; uint32_t episode = 0;
  int device = 0, n_sm = 0;
  int tile = 8;              // lanes per environment (8, 16 or 32): 32 / tile environments per warp
  uint32_t smem_entries = 0; size_t smem_bytes = 0; int grid_max = 0;
  uint32_t ring_cap = 1;     // power of two >= cap
  uint2 *d_arr = nullptr; uint32_t arr_cap = 0;      // thread-per-env kernel: arrival lists [n_envs][arr_cap] of 8-byte records (0 = none: arrivals are drawn inside the event loop)
  uint32_t arr_default = 0;  // capacity chosen at create: expected accepted arrivals per day + 8 sigma
  // mig_sim_set_prefetch: the next episode's lists are drawn in the tail of a full-day launch, into the other list buffer
  bool pf_on = false, pf_valid = false;
  uint2 *d_arr_alt = nullptr; uint32_t *d_pf_words = nullptr, *d_pf_flag = nullptr; unsigned int *d_pf_ctr = nullptr;   // ctr: {claim, finished, busy[kPfScheds]}
  uint32_t pf_pace_ns = 2000;   // measured on C5 (profiles/r2_prefetch.md): 0 / 500 / 2000 / 8000 / 32000 ns -> 72.8 / 72.6 / 72.2 / 72.4 / 72.4 ms per step
  uint32_t pf_episode = 0, pf_tag = 0;
  uint32_t envs_per_warp = 0;   // thread-per-env kernel: 0 = chosen per launch so that the batch is one resident wave
  DevTables *d_tab = nullptr;
  uint32_t *d_hdr = nullptr; uint4 *d_jobtab = nullptr; uint4 *d_dbgtab = nullptr; uint32_t *d_dbghdr = nullptr;
  unsigned int *d_counter = nullptr; uint32_t *d_algo_mask = nullptr;
  uint8_t *d_algo = nullptr, *d_cfg0 = nullptr;      // copies of the last reset's arrays (debug_trace re-runs from them)
  float *d_state = nullptr; uint8_t *d_action = nullptr;   // scratch of the DQN rollout
  uint8_t *d_table = nullptr; size_t table_bytes = 0;      // staging of rollout_host
  mig_epoch_rec_t *d_recs = nullptr; mig_totals_t *d_totals = nullptr;
  mig_job_t *d_script = nullptr; uint32_t n_script = 0;
  int epoch = -1;            // -1: never reset
  uint64_t launches = 0;
  // optional per-kernel timing (mig_sim_set_profiling): CUDA events around every launch, on the launching stream
  bool prof = false;
  struct Span { int cat; cudaEvent_t a, b; };
  std::vector<Span> spans; std::vector<cudaEvent_t> ev_pool;
};

enum { CAT_GEN = 0, CAT_SIM = 1, CAT_QNET = 2, CAT_COUNT = 3 };

// brackets one kernel launch with two events when profiling is on (otherwise free)
struct ProfSpan {
  mig_sim *s; cudaStream_t st; int cat; cudaEvent_t a = nullptr;
  static cudaEvent_t get(mig_sim *s) {
    if (!s->ev_pool.empty()) { cudaEvent_t e = s->ev_pool.back(); s->ev_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr; cudaEventCreate(&e); return e;
  }
  ProfSpan(mig_sim *s_, cudaStream_t st_, int cat_) : s(s_), st(st_), cat(cat_) { if (s->prof) { a = get(s); cudaEventRecord(a, st); } }
  ~ProfSpan() { if (a) { cudaEvent_t b = get(s); cudaEventRecord(b, st); s->spans.push_back({cat, a, b}); } }
};

// ------------------------------------------------------------------------------------------------ exact division constants
// floor(x / v) == umulhi(x, m) >> sh for every 0 <= x < 2^31 (Granlund-Montgomery, N = 31): l = ceil(log2 v),
// m = ceil(2^(31+l) / v) < 2^32, shift = l - 1.  v == 1 is flagged by sh = 32 (the quotient is x itself).
extern "C" int mig_debug_div_magic(uint32_t v, uint32_t *m, uint32_t *sh) {
  if (!m || !sh || v == 0) return fail(MIG_EINVAL, "div_magic: v must be >= 1");
  if (v == 1) { *m = 0; *sh = 32; return MIG_OK; }
  uint32_t l = 0;
  while ((1ull << l) < v) ++l;                         // l = ceil(log2 v) >= 1
  unsigned __int128 num = (unsigned __int128)1 << (31 + l);
  unsigned __int128 q = (num + v - 1) / v;
  *m = (uint32_t)q; *sh = l - 1;
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ create
static int size_index(int g) { return g == 1 ? 0 : g == 2 ? 1 : g == 3 ? 2 : g == 4 ? 3 : g == 7 ? 4 : -1; }
constexpr int kPolicyExplicit = 4;   // internal: the launch's actions come from SimArgs::actions

static int build_tables(const mig_params_t *p, DevTables *t) {
  memset(t, 0, sizeof(*t));
  if (!p->speed || !p->dur7_q || !p->class_cum || !p->slack_q10 || !p->size_at_slot || !p->accept_thr)
    return fail(MIG_EINVAL, "create: a table pointer is NULL");
  if (p->n_classes < 1 || p->n_classes > MIG_MAX_CLASSES) return fail(MIG_EINVAL, "create: n_classes %u not in 1..16", p->n_classes);
  if (p->n_configs < 1 || p->n_configs > MIG_MAX_CONFIGS) return fail(MIG_EINVAL, "create: n_configs %u not in 1..16", p->n_configs);
  if (p->cap < 1 || p->cap > 1024) return fail(MIG_EINVAL, "create: cap %u not in 1..1024", p->cap);
  if (p->epoch_s < 1 || p->n_epochs < 1 || p->n_epochs > 255) return fail(MIG_EINVAL, "create: epoch_s / n_epochs out of range");
  if (p->day_s < 0 || p->day_s > 86400) return fail(MIG_EINVAL, "create: day_s %d not in 0..86400 (one threshold per minute)", p->day_s);
  long long day_end = (long long)p->epoch_s * p->n_epochs;
  if (day_end > (1ll << 30) || p->day_s > day_end) return fail(MIG_EINVAL, "create: n_epochs * epoch_s must cover day_s and be <= 2^30");
  if (p->t_limit_s <= day_end || p->t_limit_s > (1 << 30)) return fail(MIG_EINVAL, "create: t_limit_s must be in (n_epochs*epoch_s, 2^30]");
  if (p->repart_downtime_s < 0 || p->repart_downtime_s > (1 << 24)) return fail(MIG_EINVAL, "create: repart_downtime_s out of range");
  if (p->repart_energy_mj < 0 || p->repart_energy_mj > (1ll << 48)) return fail(MIG_EINVAL, "create: repart_energy_mj out of range");
  if (p->crit_laxity_s < 0 || p->crit_laxity_s > (1 << 24)) return fail(MIG_EINVAL, "create: crit_laxity_s out of range");
  if (p->crit_max > 15) return fail(MIG_EINVAL, "create: crit_max %u > 15", p->crit_max);
  if (p->gap_scale_q16 == 0) return fail(MIG_EINVAL, "create: gap_scale_q16 must be > 0");
  for (int i = 0; i < 8; ++i) if (p->curve_mw[i] < 0 || p->curve_mw[i] > (1 << 27)) return fail(MIG_EINVAL, "create: curve_mw[%d] out of [0, 2^27]", i);
  for (int i = 0; i < 5; ++i)
    if (p->p_idle_mw[i] < 0 || p->p_idle_mw[i] > (1 << 27) || p->p_busy_mw[i] < 0 || p->p_busy_mw[i] > (1 << 27))
      return fail(MIG_EINVAL, "create: p_idle_mw / p_busy_mw[%d] out of [0, 2^27]", i);
  static const int SIZES[5] = {1, 2, 3, 4, 7};
  for (int i = 0; i < 8; ++i) t->curve[i] = p->curve_mw[i];
  for (int i = 0; i < 5; ++i) { t->p_idle[SIZES[i]] = p->p_idle_mw[i]; t->p_busy[SIZES[i]] = p->p_busy_mw[i]; }
  if (p->speed_nomig) {                                        // the MIG-disabled GPU (reading #29)
    if (p->p_idle_nomig_mw < 0 || p->p_idle_nomig_mw > (1 << 27) || p->p_busy_nomig_mw < 0 || p->p_busy_nomig_mw > (1 << 27))
      return fail(MIG_EINVAL, "create: p_idle_nomig_mw / p_busy_nomig_mw out of [0, 2^27]");
    t->p_idle[MIG_SIZE_NOMIG] = p->p_idle_nomig_mw; t->p_busy[MIG_SIZE_NOMIG] = p->p_busy_nomig_mw;
  }
  if (!(p->gamma >= 0.0f) || p->gamma > 1.0f) return fail(MIG_EINVAL, "create: gamma must be in [0, 1]");
  if (p->n_tbins || p->n_dbins || p->n_abins) {                // BINNED policy (reading #31)
    if (p->n_tbins < 1 || p->n_tbins > 255) return fail(MIG_EINVAL, "create: n_tbins %u not in 1..255", p->n_tbins);
    if (p->n_dbins < 1 || p->n_dbins > 8 || p->n_abins < 1 || p->n_abins > 8) return fail(MIG_EINVAL, "create: n_dbins / n_abins not in 1..8");
    if ((p->n_dbins > 1 && !p->dbin_edges) || (p->n_abins > 1 && !p->abin_edges)) return fail(MIG_EINVAL, "create: bin edges are NULL");
    if (p->day_s < 1) return fail(MIG_EINVAL, "create: the BINNED policy needs day_s >= 1");
    for (int i = 0; i < 8; ++i) { t->dbin_edges[i] = 0x7FFFFFFF; t->abin_edges[i] = 0x7FFFFFFF; }
    for (uint32_t i = 0; i + 1 < p->n_dbins; ++i) { if (i && p->dbin_edges[i] < p->dbin_edges[i - 1]) return fail(MIG_EINVAL, "create: dbin_edges not ascending"); t->dbin_edges[i] = p->dbin_edges[i]; }
    for (uint32_t i = 0; i + 1 < p->n_abins; ++i) { if (i && p->abin_edges[i] < p->abin_edges[i - 1]) return fail(MIG_EINVAL, "create: abin_edges not ascending"); t->abin_edges[i] = p->abin_edges[i]; }
  }
  for (uint32_t c = 0; c < p->n_configs; ++c) {
    uint32_t pack = 0; int covered_to = 0, n = 0;
    for (int s = 0; s < MIG_SLOTS; ++s) {
      int g = p->size_at_slot[c * 7 + s];
      if (!g) continue;
      if (g == MIG_SIZE_NOMIG) {                               // MIG disabled: the whole GPU, alone, at slot 0
        if (!p->speed_nomig) return fail(MIG_EINVAL, "create: config %u uses size code 8 (MIG disabled) but speed_nomig is NULL", c);
        if (s != 0 || n) return fail(MIG_EINVAL, "create: config %u: the MIG-disabled GPU must be the only slice, at slot 0", c);
        covered_to = MIG_SLOTS; pack |= (uint32_t)g << (4 * s); ++n;
        continue;
      }
      if (size_index(g) < 0) return fail(MIG_EINVAL, "create: config %u slot %d: slice size %d not in {1,2,3,4,7} (or 8 = MIG disabled)", c, s, g);
      if (s < covered_to) return fail(MIG_EINVAL, "create: config %u: slices overlap at slot %d", c, s);
      if (s + g > MIG_SLOTS) return fail(MIG_EINVAL, "create: config %u: slice at slot %d exceeds 7 slots", c, s);
      covered_to = s + g; pack |= (uint32_t)g << (4 * s); ++n;
    }
    if (!n) return fail(MIG_EINVAL, "create: config %u has no slice", c);
    t->cfg_pack[c] = pack;
    uint32_t ranks = 0, slot_of = 0; int pidle = 0;           // tie rule of reading #4: smaller size, then lower slot
    for (int s = 0; s < MIG_SLOTS; ++s) {
      int g = (pack >> (4 * s)) & 15, r = 0;
      if (!g) continue;
      for (int q = 0; q < MIG_SLOTS; ++q) { int h = (pack >> (4 * q)) & 15; if (h && (h < g || (h == g && q < s))) ++r; }
      ranks |= (uint32_t)r << (4 * s); slot_of |= (uint32_t)s << (4 * r); pidle += t->p_idle[g];
    }
    t->cfg_rank[c] = ranks; t->cfg_slot_of[c] = slot_of; t->cfg_pidle[c] = pidle;
  }
  for (uint32_t c = 0; c < p->n_classes; ++c) {
    const int32_t *q = p->dur7_q + c * 65;
    for (int i = 0; i < 65; ++i) {
      if (q[i] < 1 || q[i] > (1 << 24)) return fail(MIG_EINVAL, "create: dur7_q[%u][%d] = %d not in 1..2^24", c, i, q[i]);
      if (i && q[i] < q[i - 1]) return fail(MIG_EINVAL, "create: dur7_q[%u] not non-decreasing at %d", c, i);
      t->dur7_q[c * 65 + i] = q[i];
    }
    uint32_t vmin = 0xFFFFFFFFu, vmax = 0;
    for (int i = 0; i < 5; ++i) {
      uint32_t v = p->speed[c * 5 + i];
      if (v < 1 || v > (1u << 24)) return fail(MIG_EINVAL, "create: speed[%u][%d] = %u not in 1..2^24", c, i, v);
      vmin = v < vmin ? v : vmin; vmax = v > vmax ? v : vmax;
      uint32_t m, sh; mig_debug_div_magic(v, &m, &sh);
      t->speed[c * 5 + i] = make_uint4(v, m, sh, 0);
    }
    if (p->speed_nomig) {
      uint32_t v = p->speed_nomig[c];
      if (v < 1 || v > (1u << 24)) return fail(MIG_EINVAL, "create: speed_nomig[%u] = %u not in 1..2^24", c, v);
      vmin = v < vmin ? v : vmin; vmax = v > vmax ? v : vmax;
      uint32_t m, sh; mig_debug_div_magic(v, &m, &sh);
      t->speed_nomig[c] = make_uint4(v, m, sh, 0);
    } else t->speed_nomig[c] = t->speed[c * 5 + 4];
    unsigned long long work_max = (unsigned long long)q[64] * p->speed[c * 5 + 4];
    if (work_max + vmax >= (1ull << 31)) return fail(MIG_EINVAL, "create: class %u: max work %llu + max speed exceeds int32", c, work_max);
    if ((work_max + vmin - 1) / vmin >= (1ull << 28)) return fail(MIG_EINVAL, "create: class %u: longest duration exceeds 2^28 s", c);
    if (c && p->class_cum[c] < p->class_cum[c - 1]) return fail(MIG_EINVAL, "create: class_cum not non-decreasing at %u", c);
    t->class_cum[c] = p->class_cum[c];
    uint32_t lo = p->slack_q10[c * 2], hi = p->slack_q10[c * 2 + 1];
    if (lo > hi) return fail(MIG_EINVAL, "create: slack_q10[%u]: lo > hi", c);
    t->slack_lo[c] = lo; t->slack_span[c] = hi - lo + 1;
  }
  if (p->class_cum[p->n_classes - 1] != 0xFFFFFFFFu) return fail(MIG_EINVAL, "create: class_cum[last] must be 0xFFFFFFFF");
  for (uint32_t c = p->n_classes; c < MIG_MAX_CLASSES; ++c) t->class_cum[c] = 0xFFFFFFFFu;      // padded: the class search needs no bound
  for (int i = 0; i < MIG_THR_BINS; ++i) t->thr[i] = p->accept_thr[i];
  for (int i = 0; i <= 256; ++i) t->logT[i] = (uint32_t)llround(16777216.0 * log2(1.0 + (double)i / 256.0));
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ tile width
// Default lanes per environment: 1 = the thread-per-environment kernel, for every batch size.  Small batches put few
// environments in each warp (auto_envs_per_warp below), which makes it as fast as the 8-lane tiles where the batch cannot
// fill the machine (B200, ms per day-batch, thread kernel vs tiles: C2 1024 envs 20.6 vs 23.1, C3 4096 envs 20.9 vs 20.8,
// C4 8192 envs 31.3 vs 32.1) and 5x faster where it can (C5 65536 envs 93 vs 499).
static int default_tile(uint32_t) { return 1; }

template <bool TRACE>
static const void *kernel_ptr(int tile, bool evd = false) {
  switch (tile) {
    case 1: return evd ? (const void *)sim_thread_kernel<kThreadCta, TRACE, true> : (const void *)sim_thread_kernel<kThreadCta, TRACE, false>;
    case 8: return (const void *)sim_kernel<8, TRACE>;
    case 16: return (const void *)sim_kernel<16, TRACE>;
    default: return (const void *)sim_kernel<32, TRACE>;
  }
}

// shared-memory footprint and resident grid for `tile` lanes per environment (1 = one thread per environment)
static int configure_tile(mig_sim *s, int tile) {
  if (tile != 1 && tile != 8 && tile != 16 && tile != 32) return fail(MIG_EINVAL, "set_tile: lanes per environment must be 1, 8, 16 or 32 (got %d)", tile);
  const uint32_t cap4 = (s->p.cap + 3u) & ~3u, cap8 = (s->p.cap + 7u) & ~7u;
  uint32_t entries; size_t bytes; int threads;
  if (tile == 1) {
    // 11 ring slots of the waiting queue in shared memory per environment: 456 B per thread, 7 CTAs of 64 threads per SM = 448 resident
    // environments per SM (66 304 per B200: BASELINE C5's 65 536 run as ONE resident wave)
    entries = cap4 < 11u ? cap4 : 11u; threads = kThreadCta;
    bytes = thread_smem_bytes(entries, kThreadCta);
  } else {
    entries = cap8 < 64u ? cap8 : 64u; threads = kWarpsPerCta * 32;
    bytes = ((sizeof(HotTables) + 127) & ~(size_t)127) + (size_t)kWarpsPerCta * (32 / tile) * tile_smem_bytes(entries);
  }
  int occ = 0;
  for (int v = 0; v < (tile == 1 ? 4 : 2); ++v) {          // every instantiation that a launch may pick
    const int trace = v & 1;
    const void *k = trace ? kernel_ptr<true>(tile, v >= 2) : kernel_ptr<false>(tile, v >= 2);
    if (bytes > 48 * 1024 && cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess)
      return fail(MIG_ECUDA, "set_tile: %zu bytes of shared memory per CTA refused (%s)", bytes, cudaGetErrorString(cudaGetLastError()));
    if (tile == 1) cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    int o = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, k, threads, bytes) != cudaSuccess || o < 1)
      return fail(MIG_ECUDA, "set_tile: the rollout kernel does not fit this device (%s)", cudaGetErrorString(cudaGetLastError()));
    if (v == 0) occ = o;
  }
  if ((tile == 1) != (s->tile == 1)) s->epoch = -1;      // the saved per-env state has another layout: reset first
  s->tile = tile; s->smem_entries = entries; s->smem_bytes = bytes; s->grid_max = occ * s->n_sm;
  return MIG_OK;
}

extern "C" int mig_sim_set_tile(mig_sim_t *s, int lanes_per_env) {
  if (!s) return fail(MIG_EINVAL, "set_tile: NULL handle");
  return configure_tile(s, lanes_per_env ? lanes_per_env : default_tile(s->n_envs));
}

extern "C" int mig_sim_get_tile(const mig_sim_t *s) { return s ? s->tile : 0; }

extern "C" int mig_sim_set_envs_per_warp(mig_sim_t *s, uint32_t envs_per_warp) {
  if (!s) return fail(MIG_EINVAL, "set_envs_per_warp: NULL handle");
  if (envs_per_warp > 32 || (envs_per_warp & (envs_per_warp - 1))) return fail(MIG_EINVAL, "set_envs_per_warp: %u is not 0 or a power of two <= 32", envs_per_warp);
  s->envs_per_warp = envs_per_warp;
  return MIG_OK;
}

// (Re)allocates the arrival lists: n_envs x entries x 8 bytes, entries rounded up to a multiple of 4 (one 32-byte sector).
static int alloc_arrival_lists(mig_sim *s, uint32_t entries) {
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(MIG_ECUDA, "set_arrival_buffer: %s", cudaGetErrorString(cudaGetLastError()));
  cudaFree(s->d_arr); s->d_arr = nullptr; s->arr_cap = 0;
  cudaFree(s->d_arr_alt); s->d_arr_alt = nullptr; s->pf_valid = false;
  if (entries == 0) return MIG_OK;
  entries = (entries + 3u) & ~3u;
  const size_t need = (size_t)s->n_envs * entries * sizeof(uint2);
  if (cudaMalloc((void **)&s->d_arr, need) != cudaSuccess) {
    cudaGetLastError(); s->d_arr = nullptr;
    return fail(MIG_ENOMEM, "arrival lists: cudaMalloc of %zu bytes (%u envs x %u records x 8 B) failed; the handle now draws arrivals inside the event loop "
                            "(slower, same results) -- choose a capacity that fits with mig_sim_set_arrival_buffer", need, s->n_envs, entries);
  }
  s->arr_cap = entries;
  if (s->pf_on && cudaMalloc((void **)&s->d_arr_alt, need) != cudaSuccess) {
    cudaGetLastError(); s->d_arr_alt = nullptr; s->pf_on = false;
    return fail(MIG_ENOMEM, "arrival lists: cudaMalloc of the second buffer (%zu bytes) failed; drawing ahead is switched off", need);
  }
  return MIG_OK;
}

// Drawing ahead (off by default; results are identical either way, tested): after a full-day launch of episode e -- a
// rollout from reset under a policy that lives on the device, every environment of the handle, 32 per warp -- the warps
// that finish their day early draw the arrival lists of episode e + 1 into a second list buffer (the arrival process
// does not depend on the schedule); a following full-day launch of episode e + 1 finds them in place and
// its generator draws only what was left.  Any other call leaves the drawn lists alone (they stay valid) or, if the episode
// differs, unused.  Costs a second list buffer (n_envs x capacity x 8 bytes).
constexpr int kPfScheds = 4 * 1024;     // warp schedulers the pacing counters cover (SM id < 1024)
extern "C" int mig_sim_set_prefetch(mig_sim_t *s, int on) {
  if (!s) return fail(MIG_EINVAL, "set_prefetch: NULL handle");
  if ((on != 0) == s->pf_on) return MIG_OK;
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(MIG_ECUDA, "set_prefetch: %s", cudaGetErrorString(cudaGetLastError()));
  s->pf_valid = false;
  if (!on) { cudaFree(s->d_arr_alt); s->d_arr_alt = nullptr; s->pf_on = false; return MIG_OK; }
  if (!s->d_arr) return fail(MIG_ESTATE, "set_prefetch: the handle has no arrival lists (mig_sim_set_arrival_buffer(s, 0) was called)");
  const size_t n = s->n_envs;
  if (!s->d_pf_words) {
    if (cudaMalloc((void **)&s->d_pf_words, n * kGenWords * 4) != cudaSuccess || cudaMalloc((void **)&s->d_pf_flag, n * 4) != cudaSuccess ||
        cudaMalloc((void **)&s->d_pf_ctr, (2 + kPfScheds) * sizeof(unsigned int)) != cudaSuccess || cudaMemset(s->d_pf_flag, 0, n * 4) != cudaSuccess) {
      cudaGetLastError();
      return fail(MIG_ENOMEM, "set_prefetch: cudaMalloc failed");
    }
  }
  const size_t need = n * s->arr_cap * sizeof(uint2);
  if (cudaMalloc((void **)&s->d_arr_alt, need) != cudaSuccess) { cudaGetLastError(); s->d_arr_alt = nullptr; return fail(MIG_ENOMEM, "set_prefetch: cudaMalloc of the second list buffer (%zu bytes) failed", need); }
  s->pf_on = true;
  return MIG_OK;
}
extern "C" int mig_sim_get_prefetch(const mig_sim_t *s) { return s && s->pf_on ? 1 : 0; }

extern "C" int mig_sim_set_arrival_buffer(mig_sim_t *s, uint32_t entries_per_env) {
  if (!s) return fail(MIG_EINVAL, "set_arrival_buffer: NULL handle");
  if (entries_per_env == 0xFFFFFFFFu) entries_per_env = s->arr_default;
  if (entries_per_env > MIG_MAX_JOBS) return fail(MIG_EINVAL, "set_arrival_buffer: more than %u entries per environment", MIG_MAX_JOBS);
  return alloc_arrival_lists(s, entries_per_env);
}

extern "C" uint32_t mig_sim_get_arrival_buffer(const mig_sim_t *s) { return s ? s->arr_cap : 0; }

extern "C" int mig_sim_create(mig_sim_t **out, const mig_params_t *p, uint32_t n_envs, uint64_t seed) {
  if (!out || !p) return fail(MIG_EINVAL, "create: NULL argument");
  *out = nullptr;
  if (n_envs < 1 || n_envs > (1u << 24)) return fail(MIG_EINVAL, "create: n_envs %u not in 1..2^24", n_envs);
  std::vector<DevTables> host(1);
  int rc = build_tables(p, host.data());
  if (rc) return rc;
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev == 0) return fail(MIG_ECUDA, "create: no CUDA device (%s); there is no CPU fallback", cudaGetErrorString(ce));
  mig_sim *s = new (std::nothrow) mig_sim();
  if (!s) return fail(MIG_ENOMEM, "create: host allocation failed");
  s->p = *p;
  s->p.speed = nullptr; s->p.dur7_q = nullptr; s->p.class_cum = nullptr; s->p.slack_q10 = nullptr; s->p.size_at_slot = nullptr; s->p.accept_thr = nullptr; s->p.dbin_edges = nullptr; s->p.abin_edges = nullptr;
  if (p->speed_nomig) s->p.speed_nomig = reinterpret_cast<const uint32_t *>(1);   // (only "is it in use" is kept)
  s->n_envs = n_envs; s->seed = seed;
  cudaDeviceProp prop;
  if (cudaGetDevice(&s->device) != cudaSuccess || cudaGetDeviceProperties(&prop, s->device) != cudaSuccess) { delete s; return fail(MIG_ECUDA, "create: cannot query the device"); }
  s->n_sm = prop.multiProcessorCount;
  s->tile = 8;
  rc = configure_tile(s, default_tile(n_envs));
  if (rc) { delete s; return rc; }
  size_t n = n_envs;
#define ALLOC(ptr, bytes) if (cudaMalloc((void **)&(ptr), (bytes)) != cudaSuccess) { cudaGetLastError(); mig_sim_destroy(s); return fail(MIG_ENOMEM, "create: cudaMalloc of %zu bytes failed", (size_t)(bytes)); }
  ALLOC(s->d_tab, sizeof(DevTables));
  ALLOC(s->d_hdr, n * kHeaderWords * 4);
  s->ring_cap = 1; while (s->ring_cap < p->cap) s->ring_cap <<= 1;
  {                                                       // expected accepted arrivals per day (+ 8 sigma): capacity of an arrival list
    const double lam_max = 65536.0 * 0.6931471805599453 / (double)p->gap_scale_q16;     // candidates per second
    double acc = 0.0;
    for (int m = 0; m < MIG_THR_BINS && m * 60 < p->day_s; ++m) acc += ((double)p->accept_thr[m] + 1.0) / 4294967296.0 * lam_max * (double)((p->day_s - m * 60) < 60 ? (p->day_s - m * 60) : 60);
    double want = acc + 8.0 * sqrt(acc + 1.0) + 64.0;
    if (p->job_limit && want > (double)p->job_limit + 1.0) want = (double)p->job_limit + 1.0;
    if (want > (double)MIG_MAX_JOBS) want = (double)MIG_MAX_JOBS;
    s->arr_default = ((uint32_t)want + 7u) & ~7u;
  }
  ALLOC(s->d_jobtab, n * (s->ring_cap + kThreadTabExtra) * sizeof(uint4));
  ALLOC(s->d_dbgtab, (size_t)(s->ring_cap + kThreadTabExtra) * sizeof(uint4));
  ALLOC(s->d_dbghdr, kHeaderWords * 4);
  ALLOC(s->d_counter, sizeof(unsigned int)); ALLOC(s->d_algo_mask, sizeof(uint32_t));
  ALLOC(s->d_algo, n); ALLOC(s->d_cfg0, n);
  ALLOC(s->d_state, n * MIG_STATE_DIM * sizeof(float));
  ALLOC(s->d_action, n);
#undef ALLOC
  rc = alloc_arrival_lists(s, s->arr_default);            // a full day per environment: every launch's horizon fits
  if (rc) { mig_sim_destroy(s); return rc; }
  if (cudaMemcpy(s->d_tab, host.data(), sizeof(DevTables), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemset(s->d_hdr, 0, n * kHeaderWords * 4) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
    mig_sim_destroy(s); return fail(MIG_ECUDA, "create: table upload failed: %s", cudaGetErrorString(cudaGetLastError()));
  }
  *out = s;
  return MIG_OK;
}

extern "C" int mig_sim_destroy(mig_sim_t *s) {
  if (!s) return MIG_OK;
  cudaDeviceSynchronize();
  cudaFree(s->d_tab); cudaFree(s->d_hdr); cudaFree(s->d_jobtab); cudaFree(s->d_dbgtab); cudaFree(s->d_dbghdr); cudaFree(s->d_counter); cudaFree(s->d_algo_mask);
  cudaFree(s->d_algo); cudaFree(s->d_cfg0); cudaFree(s->d_state); cudaFree(s->d_action); cudaFree(s->d_table);
  cudaFree(s->d_recs); cudaFree(s->d_totals); cudaFree(s->d_script); cudaFree(s->d_arr); cudaFree(s->d_arr_alt); cudaFree(s->d_pf_words); cudaFree(s->d_pf_flag); cudaFree(s->d_pf_ctr);
  for (auto &sp : s->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  for (auto e : s->ev_pool) cudaEventDestroy(e);
  cudaGetLastError();
  delete s;
  return MIG_OK;
}

extern "C" uint64_t mig_sim_launch_count(const mig_sim_t *s) { return s ? s->launches : 0; }

extern "C" const char *mig_sim_kernel_name(const mig_sim_t *s) {
  if (!s) return "";
  switch (s->tile) {
    case 1: return s->p.decide_on_events ? "sim_thread_kernel<64,false,true>" : "sim_thread_kernel<64,false,false>";
    case 8: return "sim_kernel<8,false>";
    case 16: return "sim_kernel<16,false>";
    default: return "sim_kernel<32,false>";
  }
}

extern "C" int mig_sim_set_profiling(mig_sim_t *s, int on) {
  if (!s) return fail(MIG_EINVAL, "set_profiling: NULL handle");
  s->prof = on != 0;
  return MIG_OK;
}

extern "C" int mig_sim_kernel_times(mig_sim_t *s, float ms_out[3], uint32_t launches_out[3]) {
  if (!s || !ms_out) return fail(MIG_EINVAL, "kernel_times: NULL argument");
  for (int c = 0; c < CAT_COUNT; ++c) { ms_out[c] = 0.0f; if (launches_out) launches_out[c] = 0; }
  for (auto &sp : s->spans) {
    CU(cudaEventSynchronize(sp.b));
    float ms = 0.0f;
    CU(cudaEventElapsedTime(&ms, sp.a, sp.b));
    ms_out[sp.cat] += ms; if (launches_out) launches_out[sp.cat]++;
    s->ev_pool.push_back(sp.a); s->ev_pool.push_back(sp.b);
  }
  s->spans.clear();
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ launches
static void base_args(const mig_sim *s, SimArgs &a) {
  memset(&a, 0, sizeof(a));
  const mig_params_t &p = s->p;
  a.tab = s->d_tab; a.hdr = s->d_hdr; a.jobtab = s->d_jobtab; a.counter = s->d_counter;
  a.n_envs = s->n_envs; a.env_first = 0;
  a.n_classes = p.n_classes; a.n_configs = p.n_configs;
  a.k0 = (uint32_t)s->seed; a.k1 = (uint32_t)(s->seed >> 32); a.episode = s->episode; a.env_base = p.env_base;
  a.gap_scale = p.gap_scale_q16;
  a.day_s = p.day_s; a.epoch_s = p.epoch_s; a.n_epochs = p.n_epochs; a.t_limit_s = p.t_limit_s;
  a.cap = p.cap; a.job_limit = p.job_limit; a.smem_entries = s->smem_entries; a.ring_cap = s->ring_cap;
  a.downtime_s = p.repart_downtime_s; a.repart_energy = p.repart_energy_mj;
  a.theta = p.crit_laxity_s; a.crit_max = p.crit_max;
  a.w_energy = p.w_energy; a.w_tardy = p.w_tardy;
  a.algo = s->d_algo; a.cfg0 = s->d_cfg0; a.algo_mask = s->d_algo_mask;
  a.script = s->n_script ? s->d_script : nullptr; a.n_script = s->n_script;
  a.rec_stride = s->n_envs;
  a.all_down = p.repart_all_down != 0; a.util_hist = p.util_hist != 0; a.gamma = p.gamma;
  a.n_tbins = p.n_tbins; a.n_dbins = p.n_dbins; a.n_abins = p.n_abins;
}

// Environments per warp of the thread-per-env kernel: the smallest power of two that keeps the launch one resident wave
// (grid_max CTAs of kThreadCta / 32 warps): a small batch gets few environments per warp -- less serialisation of
// divergent lanes, more warps to hide latency -- and a full batch all 32 lanes.
static uint32_t auto_envs_per_warp(const mig_sim *s, uint32_t n_envs) {
  const uint64_t warps = (uint64_t)(s->grid_max > 0 ? s->grid_max : 1) * (kThreadCta / 32);
  uint32_t l = 1;
  while (l < 32 && (uint64_t)l * warps < n_envs) l <<= 1;
  return l;
}

template <bool TRACE>
static int launch_sim(mig_sim *s, const SimArgs &a, cudaStream_t st) {
  int devnow = 0;
  CU(cudaGetDevice(&devnow));
  if (devnow != s->device) return fail(MIG_ESTATE, "the simulator lives on device %d but device %d is current: its pointers are not valid here", s->device, devnow);
  if (s->tile == 1) {                                     // one thread per environment, one CTA per 64 environments
    SimArgs b = a;
    // arrivals of this launch's horizon: drawn by the generator kernel into the per-environment lists, on the same stream,
    // before the event loop runs (not for scripted arrivals, nor for the one-env debug trace, which draws its own)
    const bool lists = s->d_arr && a.n_steps > 0 && !a.script && !a.from_init && !a.hdr_override;
    // a full day of every environment of the handle, straight from reset: the launch whose lists may have been drawn ahead
    // (mig_sim_set_prefetch) and whose tail draws the next episode's
    const bool full_day = lists && !TRACE && s->pf_on && s->d_arr_alt && s->epoch == 0 && a.n_steps >= a.n_epochs && a.env_first == 0 && a.n_envs == s->n_envs;
    if (lists) {
      GenArgs g; memset(&g, 0, sizeof(g));
      if (full_day && s->pf_valid && s->pf_episode == a.episode) {      // drawn ahead: the lists are in the other buffer
        std::swap(s->d_arr, s->d_arr_alt);
        g.pf_flag = s->d_pf_flag; g.pf_words = s->d_pf_words; g.pf_tag = s->pf_tag;
      }
      if (full_day) s->pf_valid = false;
      g.tab = a.tab; g.hdr = a.hdr; g.arr = s->d_arr; g.arr_cap = s->arr_cap; g.n_envs = a.n_envs; g.env_first = a.env_first;
      g.k0 = a.k0; g.k1 = a.k1; g.episode = a.episode; g.env_base = a.env_base; g.gap_scale = a.gap_scale;
      g.day_s = a.day_s; g.epoch_s = a.epoch_s; g.n_epochs = a.n_epochs; g.n_steps = a.n_steps; g.job_limit = a.job_limit;
      { ProfSpan ps(s, st, CAT_GEN); gen_arrivals_kernel<<<(a.n_envs + kGenWarps - 1) / kGenWarps, kGenWarps * 32, 0, st>>>(g); }
      CU(cudaGetLastError());
      s->launches++;
    }
    b.arr = lists ? s->d_arr : nullptr; b.arr_cap = s->arr_cap;
    b.envs_per_warp = s->envs_per_warp ? s->envs_per_warp : auto_envs_per_warp(s, b.n_envs);
    if (full_day && b.envs_per_warp == 32u && b.n_envs >= 32u) {        // the launch's tail draws episode + 1 into the other buffer
      CU(cudaMemsetAsync(s->d_pf_ctr, 0, (2 + kPfScheds) * sizeof(unsigned int), st));
      b.pf_on = 1;
      PrefetchArgs &pf = b.pf;
      pf.g.tab = a.tab; pf.g.hdr = nullptr; pf.g.arr = s->d_arr_alt; pf.g.arr_cap = s->arr_cap; pf.g.n_envs = s->n_envs; pf.g.env_first = 0;
      pf.g.k0 = a.k0; pf.g.k1 = a.k1; pf.g.episode = a.episode + 1u; pf.g.env_base = a.env_base; pf.g.gap_scale = a.gap_scale;
      pf.g.day_s = a.day_s; pf.g.epoch_s = a.epoch_s; pf.g.n_epochs = a.n_epochs; pf.g.n_steps = a.n_epochs; pf.g.job_limit = a.job_limit;
      pf.g.pf_flag = nullptr; pf.g.pf_words = nullptr; pf.g.pf_tag = 0;
      pf.words = s->d_pf_words; pf.flag = s->d_pf_flag; pf.tag = ++s->pf_tag;
      if (pf.tag == 0) pf.tag = ++s->pf_tag;                            // (0 is the flags' initial value)
      pf.claim = s->d_pf_ctr; pf.finished = s->d_pf_ctr + 1; pf.n_warps = b.n_envs / 32u;
      pf.busy = s->d_pf_ctr + 2; pf.pace_ns = s->pf_pace_ns;
      s->pf_valid = true; s->pf_episode = a.episode + 1u;
    }
    const uint32_t per_cta = b.envs_per_warp * (kThreadCta / 32);
    const dim3 grid((b.n_envs + per_cta - 1) / per_cta), block(kThreadCta);
    {
      ProfSpan ps(s, st, CAT_SIM);
      if (b.ev_decide) sim_thread_kernel<kThreadCta, TRACE, true><<<grid, block, s->smem_bytes, st>>>(b);
      else sim_thread_kernel<kThreadCta, TRACE, false><<<grid, block, s->smem_bytes, st>>>(b);
    }
    CU(cudaGetLastError());
    s->launches++;
    return MIG_OK;
  }
  CU(cudaMemsetAsync(s->d_counter, 0, sizeof(unsigned int), st));
  const uint32_t envs_per_cta = (uint32_t)kWarpsPerCta * (32u / (uint32_t)s->tile);
  int ctas = (int)((a.n_envs + envs_per_cta - 1) / envs_per_cta);
  if (ctas > s->grid_max) ctas = s->grid_max;
  const dim3 grid((unsigned)ctas), block(kWarpsPerCta * 32);
  {
    ProfSpan ps(s, st, CAT_SIM);
    switch (s->tile) {
      case 8: sim_kernel<8, TRACE><<<grid, block, s->smem_bytes, st>>>(a); break;
      case 16: sim_kernel<16, TRACE><<<grid, block, s->smem_bytes, st>>>(a); break;
      default: sim_kernel<32, TRACE><<<grid, block, s->smem_bytes, st>>>(a); break;
    }
  }
  CU(cudaGetLastError());
  s->launches++;
  return MIG_OK;
}

extern "C" int mig_sim_reset(mig_sim_t *s, uint32_t episode, const uint8_t *algo, const uint8_t *cfg0, float *state_out, void *stream) {
  if (!s || !algo || !cfg0) return fail(MIG_EINVAL, "reset: NULL argument");
  cudaStream_t st = (cudaStream_t)stream;
  CU(cudaMemcpyAsync(s->d_algo, algo, s->n_envs, cudaMemcpyDeviceToDevice, st));
  CU(cudaMemcpyAsync(s->d_cfg0, cfg0, s->n_envs, cudaMemcpyDeviceToDevice, st));
  s->episode = episode;
  CU(cudaMemsetAsync(s->d_algo_mask, 0, sizeof(uint32_t), st));     // (the init launch collects the batch's algorithms)
  SimArgs a; base_args(s, a);
  a.from_init = 1; a.save = 1; a.n_steps = 0; a.state_out = state_out;
  int rc = launch_sim<false>(s, a, st);
  if (rc) return rc;
  s->epoch = 0;
  return MIG_OK;
}

extern "C" int mig_sim_step(mig_sim_t *s, const uint8_t *action, float *state_out, float *reward_out, int64_t *energy_mj_out,
                            int64_t *tardiness_s_out, mig_epoch_rec_t *rec_out, mig_epoch_rec_t *drain_rec_out, void *stream) {
  if (!s || !action) return fail(MIG_EINVAL, "step: NULL argument");
  if (s->epoch < 0) return fail(MIG_ESTATE, "step: reset has not been called");
  if (s->epoch >= s->p.n_epochs) return fail(MIG_ESTATE, "step: the day is over (%d epochs done); call reset", s->epoch);
  SimArgs a; base_args(s, a);
  a.save = 1; a.n_steps = 1; a.policy = kPolicyExplicit;
  a.actions = action; a.act_stride_env = 1; a.act_stride_k = 0;
  a.state_out = state_out; a.reward_out = reward_out; a.energy_out = energy_mj_out; a.tard_out = tardiness_s_out;
  a.recs = rec_out; a.rec_k0 = s->epoch; a.drain_rec = drain_rec_out;
  int rc = launch_sim<false>(s, a, (cudaStream_t)stream);
  if (rc) return rc;
  s->epoch++;
  return MIG_OK;
}

static int launch_qnet(const mig_qnet *q, QArgs &qa, cudaStream_t st) {
  qa.W1 = q->W1; qa.b1 = q->b1; qa.W2 = q->W2; qa.b2 = q->b2; qa.W3 = q->W3; qa.b3 = q->b3; qa.H = q->H; qa.A = q->A;
  size_t smem = (size_t)(MIG_STATE_DIM + 2 * q->H + q->A) * kQRows * sizeof(float) + (size_t)kQStages * kQChunk * q->H * sizeof(float);
  static size_t attr_set[64] = {0};            // per DEVICE: the opt-in to > 48 KB of dynamic shared memory is a per-device function attribute
  int devnow = 0;
  CU(cudaGetDevice(&devnow));
  if (devnow != q->device) return fail(MIG_ESTATE, "q_eval: the Q-network lives on device %d but device %d is current", q->device, devnow);
  if (smem > 48 * 1024 && (devnow < 0 || devnow >= 64 || attr_set[devnow] < smem)) {
    CU(cudaFuncSetAttribute(qnet_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (devnow >= 0 && devnow < 64) attr_set[devnow] = smem;
  }
  uint32_t blocks = (qa.B + kQRows - 1) / kQRows;
  qnet_kernel<<<blocks, q->H / kQCols * (kQRows / kQRpt), smem, st>>>(qa);
  CU(cudaGetLastError());
  return MIG_OK;
}

extern "C" int mig_sim_rollout(mig_sim_t *s, int policy, const uint8_t *table, const mig_qnet_t *q, float epsilon,
                               mig_epoch_rec_t *recs_out, mig_totals_t *totals_out, void *stream) {
  if (!s) return fail(MIG_EINVAL, "rollout: NULL handle");
  if (s->epoch < 0) return fail(MIG_ESTATE, "rollout: reset has not been called");
  if (s->epoch >= s->p.n_epochs) return fail(MIG_ESTATE, "rollout: the day is over; call reset");
  if (policy != MIG_POLICY_STATIC && policy != MIG_POLICY_TABLE && policy != MIG_POLICY_DQN && policy != MIG_POLICY_BINNED) return fail(MIG_EINVAL, "rollout: unknown policy %d", policy);
  if ((policy == MIG_POLICY_TABLE || policy == MIG_POLICY_BINNED) && !table) return fail(MIG_EINVAL, "rollout: TABLE / BINNED policy needs a table");
  if (policy == MIG_POLICY_BINNED && !s->p.n_tbins) return fail(MIG_EINVAL, "rollout: the BINNED policy needs n_tbins / n_dbins / n_abins at create");
  cudaStream_t st = (cudaStream_t)stream;
  const int ne = s->p.n_epochs;
  if (policy != MIG_POLICY_DQN) {
    SimArgs a; base_args(s, a);
    a.save = 1; a.n_steps = ne - s->epoch; a.policy = policy;
    if (policy == MIG_POLICY_BINNED) a.bin_table = table; else a.table = table;
    a.ev_decide = (policy == MIG_POLICY_TABLE || policy == MIG_POLICY_BINNED) && s->p.decide_on_events;
    a.recs = recs_out; a.rec_k0 = 0; a.drain_rec = recs_out ? recs_out + (size_t)ne * s->n_envs : nullptr;
    a.totals = totals_out;
    int rc = launch_sim<false>(s, a, st);
    if (rc) return rc;
    s->epoch = ne;
    return MIG_OK;
  }
  if (!q) return fail(MIG_EINVAL, "rollout: DQN policy needs a Q-network");
  if (q->A != s->p.n_configs) return fail(MIG_EINVAL, "rollout: Q-network has %u actions, the simulator %u configurations", q->A, s->p.n_configs);
  if (!(epsilon >= 0.0f) || epsilon > 1.0f) return fail(MIG_EINVAL, "rollout: epsilon must be in [0, 1]");
  double et = (double)epsilon * 4294967296.0;
  uint32_t eps_thr = et >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)llround(et);
  {                                             // current observation into the handle's scratch
    SimArgs a; base_args(s, a);
    a.save = 0; a.n_steps = 0; a.state_out = s->d_state;
    int rc = launch_sim<false>(s, a, st);
    if (rc) return rc;
  }
  while (s->epoch < ne) {
    QArgs qa; memset(&qa, 0, sizeof(qa));
    qa.state = s->d_state; qa.B = s->n_envs; qa.action_out = s->d_action; qa.eps_thr = eps_thr;
    qa.epoch = (uint32_t)s->epoch; qa.k0 = (uint32_t)s->seed; qa.k1 = (uint32_t)(s->seed >> 32); qa.episode = s->episode; qa.env_base = s->p.env_base;
    int rc;
    { ProfSpan ps(s, st, CAT_QNET); rc = launch_qnet(q, qa, st); }
    if (rc) return rc;
    s->launches++;
    SimArgs a; base_args(s, a);
    a.save = 1; a.n_steps = 1; a.policy = kPolicyExplicit;
    a.actions = s->d_action; a.act_stride_env = 1; a.act_stride_k = 0;
    a.state_out = s->d_state;
    a.recs = recs_out; a.rec_k0 = 0; a.drain_rec = recs_out ? recs_out + (size_t)ne * s->n_envs : nullptr;
    if (s->epoch == ne - 1) a.totals = totals_out;
    rc = launch_sim<false>(s, a, st);
    if (rc) return rc;
    s->epoch++;
  }
  return MIG_OK;
}

extern "C" int mig_sim_totals(mig_sim_t *s, mig_totals_t *totals_out, void *stream) {
  if (!s || !totals_out) return fail(MIG_EINVAL, "totals: NULL argument");
  if (s->epoch < 0) return fail(MIG_ESTATE, "totals: reset has not been called");
  SimArgs a; base_args(s, a);
  a.save = 0; a.n_steps = 0; a.totals = totals_out;
  return launch_sim<false>(s, a, (cudaStream_t)stream);
}

extern "C" int mig_sim_aux(mig_sim_t *s, float *return_out, int32_t *util_s_out, void *stream) {
  if (!s) return fail(MIG_EINVAL, "aux: NULL handle");
  if (s->epoch < 0) return fail(MIG_ESTATE, "aux: reset has not been called");
  if (util_s_out && !s->p.util_hist) return fail(MIG_ESTATE, "aux: params.util_hist was 0 at create: the utilisation levels were not kept");
  if (!return_out && !util_s_out) return MIG_OK;
  aux_kernel<<<(s->n_envs + 255) / 256, 256, 0, (cudaStream_t)stream>>>(s->d_hdr, s->n_envs, s->tile != 1, return_out, util_s_out);
  CU(cudaGetLastError());
  s->launches++;
  return MIG_OK;
}

// ET: host reduction in double; a = t / (2 s) from the GLOBAL means
extern "C" int mig_et_reduce(const double *x, const double *y, const uint32_t *group, uint32_t n, uint32_t n_groups, double *et_out, double *a_out) {
  if (!x || !y || !group || !et_out || n == 0 || n_groups == 0) return fail(MIG_EINVAL, "et_reduce: NULL argument or n = 0");
  double sx = 0.0, sy = 0.0;
  for (uint32_t i = 0; i < n; ++i) { if (group[i] >= n_groups) return fail(MIG_EINVAL, "et_reduce: group[%u] = %u out of range", i, group[i]); sx += x[i]; sy += y[i]; }
  const double smean = sx / n, tmean = sy / n;
  if (!(smean > 0.0)) return fail(MIG_EINVAL, "et_reduce: the mean energy must be positive");
  const double a = tmean / (2.0 * smean);
  std::vector<double> acc(n_groups, 0.0); std::vector<uint32_t> cnt(n_groups, 0);
  for (uint32_t i = 0; i < n; ++i) { acc[group[i]] += (a * x[i] + y[i]) / (a + 1.0); cnt[group[i]]++; }
  for (uint32_t g = 0; g < n_groups; ++g) et_out[g] = cnt[g] ? acc[g] / cnt[g] : 0.0;
  if (a_out) *a_out = a;
  return MIG_OK;
}

// The device's address of a HOST buffer that it can write directly -- pinned and mapped memory (cudaHostAlloc,
// cudaHostRegister) -- or NULL for ordinary host memory.  First and last byte are looked up: both must be registered.
static void *mapped_device_ptr(const void *host, size_t bytes) {
  cudaPointerAttributes lo, hi;
  if (!host || bytes == 0) return nullptr;
  if (cudaPointerGetAttributes(&lo, host) != cudaSuccess || cudaPointerGetAttributes(&hi, static_cast<const char *>(host) + bytes - 1) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  if (lo.type != cudaMemoryTypeHost || hi.type != cudaMemoryTypeHost || !lo.devicePointer) return nullptr;
  return lo.devicePointer;
}

extern "C" int mig_sim_rollout_host(mig_sim_t *s, uint32_t episode, const uint8_t *algo, const uint8_t *cfg0, int policy,
                                    const uint8_t *table, const mig_qnet_t *q, float epsilon, mig_epoch_rec_t *recs_out,
                                    mig_totals_t *totals_out) {
  if (!s || !algo || !cfg0 || !totals_out) return fail(MIG_EINVAL, "rollout_host: NULL argument");
  const size_t n = s->n_envs, ne = (size_t)s->p.n_epochs;
  // result buffers in pinned, mapped host memory are written by the kernels themselves (every record and every totals row
  // is stored once, 64 and 80 contiguous bytes per environment): the results cross the link while the launch runs and
  // there is no copy after it; ordinary host memory goes through the handle's device copy
  mig_totals_t *tot_map = static_cast<mig_totals_t *>(mapped_device_ptr(totals_out, n * sizeof(mig_totals_t)));
  mig_epoch_rec_t *rec_map = static_cast<mig_epoch_rec_t *>(mapped_device_ptr(recs_out, recs_out ? n * (ne + 1) * sizeof(mig_epoch_rec_t) : 0));
  if (!tot_map && !s->d_totals) { if (cudaMalloc((void **)&s->d_totals, n * sizeof(mig_totals_t)) != cudaSuccess) { cudaGetLastError(); return fail(MIG_ENOMEM, "rollout_host: cudaMalloc failed"); } }
  if (recs_out && !rec_map && !s->d_recs) { if (cudaMalloc((void **)&s->d_recs, n * (ne + 1) * sizeof(mig_epoch_rec_t)) != cudaSuccess) { cudaGetLastError(); return fail(MIG_ENOMEM, "rollout_host: cudaMalloc failed"); } }
  if (policy == MIG_POLICY_TABLE || policy == MIG_POLICY_BINNED) {
    if (!table) return fail(MIG_EINVAL, "rollout_host: TABLE / BINNED policy needs a table");
    const size_t Bc = 1 + (size_t)s->p.n_dbins * s->p.n_abins;
    size_t tb = policy == MIG_POLICY_TABLE ? n * ne * 4 : (size_t)s->p.n_configs * s->p.n_tbins * Bc * Bc * Bc;
    if (s->table_bytes < tb) { cudaFree(s->d_table); s->d_table = nullptr; if (cudaMalloc((void **)&s->d_table, tb) != cudaSuccess) { cudaGetLastError(); s->table_bytes = 0; return fail(MIG_ENOMEM, "rollout_host: cudaMalloc failed"); } s->table_bytes = tb; }
    CU(cudaMemcpyAsync(s->d_table, table, tb, cudaMemcpyHostToDevice, 0));
  }
  // reset() copies device -> device from its arguments: stage the host arrays in the DQN action/state scratch first
  uint8_t *stage_algo = s->d_action; uint8_t *stage_cfg = reinterpret_cast<uint8_t *>(s->d_state);
  CU(cudaMemcpyAsync(stage_algo, algo, n, cudaMemcpyHostToDevice, 0));
  CU(cudaMemcpyAsync(stage_cfg, cfg0, n, cudaMemcpyHostToDevice, 0));
  int rc = mig_sim_reset(s, episode, stage_algo, stage_cfg, nullptr, nullptr);
  if (rc) return rc;
  rc = mig_sim_rollout(s, policy, s->d_table, q, epsilon, recs_out ? (rec_map ? rec_map : s->d_recs) : nullptr, tot_map ? tot_map : s->d_totals, nullptr);
  if (rc) return rc;
  if (!tot_map) CU(cudaMemcpyAsync(totals_out, s->d_totals, n * sizeof(mig_totals_t), cudaMemcpyDeviceToHost, 0));
  if (recs_out && !rec_map) CU(cudaMemcpyAsync(recs_out, s->d_recs, n * (ne + 1) * sizeof(mig_epoch_rec_t), cudaMemcpyDeviceToHost, 0));
  CU(cudaStreamSynchronize(0));
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ Q-network
extern "C" int mig_qnet_create(mig_qnet_t **out, const float *W1, const float *b1, const float *W2, const float *b2,
                               const float *W3, const float *b3, uint32_t hidden, uint32_t n_actions) {
  if (!out || !W1 || !b1 || !W2 || !b2 || !W3 || !b3) return fail(MIG_EINVAL, "qnet_create: NULL argument");
  *out = nullptr;
  if (hidden < 32 || hidden > 256 || hidden % 32) return fail(MIG_EINVAL, "qnet_create: hidden %u must be a multiple of 32 in 32..256", hidden);
  if (n_actions < 1 || n_actions > MIG_MAX_CONFIGS) return fail(MIG_EINVAL, "qnet_create: n_actions %u not in 1..16", n_actions);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(MIG_ECUDA, "qnet_create: no CUDA device; there is no CPU fallback"); }
  mig_qnet *q = new (std::nothrow) mig_qnet();
  if (!q) return fail(MIG_ENOMEM, "qnet_create: host allocation failed");
  const size_t H = hidden, A = n_actions;
  const size_t sz[6] = {MIG_STATE_DIM * H, H, H * H, H, H * A, A};
  const float *src[6] = {W1, b1, W2, b2, W3, b3};
  size_t off[6], tot = 0;
  for (int i = 0; i < 6; ++i) { off[i] = tot; tot += (sz[i] + 3) & ~(size_t)3; }
  if (cudaMalloc((void **)&q->d, tot * sizeof(float)) != cudaSuccess) { cudaGetLastError(); delete q; return fail(MIG_ENOMEM, "qnet_create: cudaMalloc failed"); }
  for (int i = 0; i < 6; ++i)
    if (cudaMemcpy(q->d + off[i], src[i], sz[i] * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(q->d); delete q; return fail(MIG_ECUDA, "qnet_create: upload failed"); }
  q->W1 = q->d + off[0]; q->b1 = q->d + off[1]; q->W2 = q->d + off[2]; q->b2 = q->d + off[3]; q->W3 = q->d + off[4]; q->b3 = q->d + off[5];
  q->H = hidden; q->A = n_actions;
  cudaGetDevice(&q->device);
  *out = q;
  return MIG_OK;
}

extern "C" int mig_qnet_destroy(mig_qnet_t *q) {
  if (!q) return MIG_OK;
  cudaDeviceSynchronize(); cudaFree(q->d); cudaGetLastError();
  delete q;
  return MIG_OK;
}

extern "C" int mig_q_eval(const mig_qnet_t *q, const float *state, uint32_t B, float *q_out, uint8_t *argmax_out, void *stream) {
  if (!q || !state) return fail(MIG_EINVAL, "q_eval: NULL argument");
  if (B == 0) return MIG_OK;
  QArgs qa; memset(&qa, 0, sizeof(qa));
  qa.state = state; qa.B = B; qa.q_out = q_out; qa.argmax_out = argmax_out;
  return launch_qnet(q, qa, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------ debug / parity
extern "C" int mig_sim_debug_trace(mig_sim_t *s, uint32_t env, int policy, const uint8_t *table, const uint8_t *actions,
                                   mig_event_t *buf, uint32_t cap_events, uint32_t *n_out, mig_totals_t *totals_out, void *stream) {
  if (!s || !n_out) return fail(MIG_EINVAL, "debug_trace: NULL argument");
  if (s->epoch < 0) return fail(MIG_ESTATE, "debug_trace: reset has not been called");
  if (env >= s->n_envs) return fail(MIG_EINVAL, "debug_trace: env %u out of range", env);
  if (!actions && policy != MIG_POLICY_STATIC && policy != MIG_POLICY_TABLE && policy != MIG_POLICY_BINNED) return fail(MIG_EINVAL, "debug_trace: policy must be STATIC, TABLE or BINNED, or pass actions");
  if (!actions && policy != MIG_POLICY_STATIC && !table) return fail(MIG_EINVAL, "debug_trace: TABLE / BINNED policy needs a table");
  if (!actions && policy == MIG_POLICY_BINNED && !s->p.n_tbins) return fail(MIG_EINVAL, "debug_trace: the BINNED policy needs n_tbins / n_dbins / n_abins at create");
  SimArgs a; base_args(s, a);
  a.n_envs = 1; a.env_first = env; a.tab_override = s->d_dbgtab; a.hdr_override = s->d_dbghdr;
  a.from_init = 1; a.save = 0; a.n_steps = s->p.n_epochs;
  if (actions) { a.policy = kPolicyExplicit; a.actions = actions; a.act_stride_env = 0; a.act_stride_k = 1; }
  else {
    a.policy = policy;
    if (policy == MIG_POLICY_BINNED) a.bin_table = table; else a.table = table;
    a.ev_decide = policy != MIG_POLICY_STATIC && s->p.decide_on_events;
  }
  a.trace = buf; a.trace_cap = buf ? cap_events : 0; a.trace_n = n_out; a.totals = totals_out;
  return launch_sim<true>(s, a, (cudaStream_t)stream);
}

extern "C" int mig_sim_debug_set_jobs(mig_sim_t *s, const mig_job_t *jobs, uint32_t n) {
  if (!s) return fail(MIG_EINVAL, "debug_set_jobs: NULL handle");
  CU(cudaDeviceSynchronize());
  cudaFree(s->d_script); s->d_script = nullptr; s->n_script = 0;
  if (n == 0) return MIG_OK;
  if (!jobs) return fail(MIG_EINVAL, "debug_set_jobs: NULL jobs");
  if (n > MIG_MAX_JOBS) return fail(MIG_EINVAL, "debug_set_jobs: too many jobs");
  std::vector<DevTables> host(1);
  CU(cudaMemcpy(host.data(), s->d_tab, sizeof(DevTables), cudaMemcpyDeviceToHost));
  for (uint32_t i = 0; i < n; ++i) {
    const mig_job_t &j = jobs[i];
    if (j.cls >= s->p.n_classes) return fail(MIG_EINVAL, "debug_set_jobs: job %u: class %u out of range", i, j.cls);
    if (j.arr < 0 || j.arr > (1 << 30) || j.due < 0 || j.due > (1 << 30)) return fail(MIG_EINVAL, "debug_set_jobs: job %u: arr/due out of [0, 2^30]", i);
    if (i && j.arr < jobs[i - 1].arr) return fail(MIG_EINVAL, "debug_set_jobs: arrivals must be non-decreasing (job %u)", i);
    if (j.dur7 < 1 || j.dur7 > (1 << 24)) return fail(MIG_EINVAL, "debug_set_jobs: job %u: dur7 %d not in 1..2^24", i, j.dur7);
    uint32_t vmin = 0xFFFFFFFFu, vmax = 0;
    for (int k = 0; k < 5; ++k) { uint32_t v = host[0].speed[j.cls * 5 + k].x; vmin = v < vmin ? v : vmin; vmax = v > vmax ? v : vmax; }
    { uint32_t v = host[0].speed_nomig[j.cls].x; vmin = v < vmin ? v : vmin; vmax = v > vmax ? v : vmax; }
    unsigned long long work = (unsigned long long)j.dur7 * host[0].speed[j.cls * 5 + 4].x;
    if (work + vmax >= (1ull << 31) || (work + vmin - 1) / vmin >= (1ull << 28))
      return fail(MIG_EINVAL, "debug_set_jobs: job %u: work %llu out of the int32 / 2^28 s range", i, work);
  }
  if (cudaMalloc((void **)&s->d_script, (size_t)n * sizeof(mig_job_t)) != cudaSuccess) { cudaGetLastError(); return fail(MIG_ENOMEM, "debug_set_jobs: cudaMalloc failed"); }
  CU(cudaMemcpy(s->d_script, jobs, (size_t)n * sizeof(mig_job_t), cudaMemcpyHostToDevice));
  s->n_script = n;
  return MIG_OK;
}
