// sim_device.cuh -- the rollout kernel: ONE WARP TILE OF G LANES PER ENVIRONMENT (G = 8, 16 or 32; 32 / G environments
// per warp run in lockstep).  north_star (a) names one warp per environment; the measured queues of the paper-shaped
// workloads are short (a dozen jobs) and a MIG GPU has 7 slots, so 8 lanes hold a whole environment and a warp carries
// four of them per instruction.  G = 32 is the north-star layout and stays selectable.
//
// Each tile simulates one MIG-partitioned GPU through `n_steps` decision epochs, event by event
// (every arrival / completion is a preemption point at which ALL jobs in the system are re-evaluated).
//   * job table {skey, meta | rem, due} (16 B / job, two 8-byte arrays) in shared memory, overflow in global;
//   * slice table: tile lane p < 7 owns the slice that starts at slot p (size, down/up, running job cached in registers);
//   * reschedule = up to 7 tile-argmin passes over the priority key (butterfly SHFL, or REDUX at G = 32, + ballot), slice
//     choice by the 7 slice lanes in parallel (one exact magic-number division each), PREEMPT/START diff;
//   * arrivals: counter-based Philox4x32-10, G thinning candidates per pass (one per lane), gaps prefix-summed in 64-bit
//     fixed point (integer => associative => identical to sequential accumulation);
//   * energy / tardiness in int64, trace hash FNV-1a-64 over every event.
// Control flow is WARP-UNIFORM wherever a cross-lane primitive is executed (every SHFL / VOTE / REDUX uses the full
// mask; per-tile activity is a predicate): run-time member masks cost a WARPSYNC.COLLECTIVE round trip (measured 300+
// cycles on B200), full-mask segmented shuffles cost one instruction.
// All readings (tie rules, same-tick order, drain, ...) are DESIGN.md section 3.  No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>

#include "philox.cuh"
#include "sim_common.h"

namespace migsim {

#define MIG_FULL 0xffffffffu
#define MIG_INF 0x7fffffff
#define MIG_NOJOB 0xFFFFFFFFu

// counters of a record span; counter c lives on tile lane c % G of register cntA (c < G) or cntB (c >= G)
enum { C_ARRIVED = 0, C_COMPLETED, C_DROPPED, C_TARDY, C_PREEMPT, C_START, C_CRIT, C_EVENTS, C_REPART, C_SYSMAX, C_COUNT };   // = word order of mig_totals_t

// per-tile scratch in shared memory (words): a 64-word staging area (header / record / state vector), the totals
enum { WS_STAGE = 0, WS_CNT = 64, WS_TOT = 74 /* 3 x u64 */, WS_TBASE = 80 /* u64 */, WS_DROPS = 82, WS_WORDS = 96 };

// saved per-env header (kHeaderWords words, a.hdr): word indices
enum { H_UPAT = 0 /* 7 */, H_T = 7, H_PK, H_NSYS, H_HLO, H_HHI, H_GKBASE, H_TBASE_LO, H_TBASE_HI, H_GPENDING, H_NACC, H_GDONE,
       H_ISCRIPT, H_DROPS, H_TOT /* 6 */, H_LOOKV = 26, H_LOOKTICK, H_LOOKCLS, H_LOOKWORK, H_LOOKDUE, H_LOOKID,
       H_SLICE = 32 /* 7 */, H_GK = 39, H_GT_LO, H_GT_HI, H_UTIL_HI = 42 /* 2: utilisation levels 6, 7 */,
       H_RET = 44 /* discounted return so far, fp32 bits */, H_DISC /* gamma^k, fp32 bits */, H_CNT = 48 /* 10 */,
       H_UTIL_LO = 58 /* 6: seconds at utilisation levels 0..5 */ };
__host__ __device__ constexpr int tile_util_word(int level) { return level < 6 ? H_UTIL_LO + level : H_UTIL_HI + level - 6; }

struct HotTables {               // per CTA, shared memory
  uint4 speed[MIG_MAX_CLASSES * 5];
  uint4 speed_nomig[MIG_MAX_CLASSES];   // size code 8: the whole GPU with MIG disabled (reading #29)
  uint32_t cfg_pack[MIG_MAX_CONFIGS];
  int32_t curve[8], p_idle[12], p_busy[12];
};

__host__ __device__ constexpr size_t tile_smem_bytes(uint32_t smem_entries) {
  // scratch + two 8-byte arrays; + 64 so that consecutive tiles start 64 B apart modulo 128 (LDS.64 of two tiles = one wavefront)
  return (size_t)WS_WORDS * 4 + (size_t)smem_entries * 16 + 64;
}

__device__ __forceinline__ int sidx_of(int size) { return size == 7 ? 4 : size - 1; }   // 1,2,3,4,7 -> 0..4
__device__ __forceinline__ int tile_units_of(int size) { return min(size, 7); }         // compute units: size code 8 is the whole GPU

// ceil(rem / v) for 0 < rem, rem + v - 1 < 2^31, by the precomputed magic number of v (exact; see mig_debug_div_magic)
__device__ __forceinline__ int rd_magic(int rem, uint4 sp) {
  uint32_t x = (uint32_t)rem + sp.x - 1u;
  uint32_t q = __umulhi(x, sp.y) >> (sp.z & 31u);
  return (int)(sp.z >= 32u ? x : q);
}

// ---------------------------------------------------------------------------------------------- tile primitives
// Every function is executed by all 32 lanes (full mask); results are per tile of G lanes.
template <int G>
struct Tile {
  static_assert(G == 8 || G == 16 || G == 32, "tile width");
  static __device__ __forceinline__ int tmin(int v) {
    if constexpr (G == 32) return __reduce_min_sync(MIG_FULL, v);
    else {
#pragma unroll
      for (int d = G / 2; d; d >>= 1) v = min(v, __shfl_xor_sync(MIG_FULL, v, d));
      return v;
    }
  }
  static __device__ __forceinline__ int tmax(int v) {
    if constexpr (G == 32) return __reduce_max_sync(MIG_FULL, v);
    else {
#pragma unroll
      for (int d = G / 2; d; d >>= 1) v = max(v, __shfl_xor_sync(MIG_FULL, v, d));
      return v;
    }
  }
  static __device__ __forceinline__ uint32_t tminu(uint32_t v) {
    if constexpr (G == 32) return __reduce_min_sync(MIG_FULL, v);
    else {
#pragma unroll
      for (int d = G / 2; d; d >>= 1) v = min(v, __shfl_xor_sync(MIG_FULL, v, d));
      return v;
    }
  }
  static __device__ __forceinline__ int tadd(int v) {
    if constexpr (G == 32) return __reduce_add_sync(MIG_FULL, v);
    else {
#pragma unroll
      for (int d = G / 2; d; d >>= 1) v += __shfl_xor_sync(MIG_FULL, v, d);
      return v;
    }
  }
  // ballot restricted to the caller's tile, bit i = tile lane i
  static __device__ __forceinline__ uint32_t tballot(bool p, int gshift) {
    uint32_t b = __ballot_sync(MIG_FULL, p);
    if constexpr (G == 32) return b;
    else return (b >> gshift) & ((1u << G) - 1u);
  }
  template <typename T>
  static __device__ __forceinline__ T tshfl(T v, int src) { return __shfl_sync(MIG_FULL, v, src, G); }   // src = tile lane
};

#define MIG_ANY(p) __any_sync(MIG_FULL, (p))

template <int G, bool TRACE>
struct Env {
  using T = Tile<G>;
  // ------------------------------------------------------------------ environment state (registers)
  const SimArgs &a;
  const HotTables &hot;
  uint32_t *ws;            // this tile's scratch (shared)
  uint2 *skm, *srd;        // this tile's job table (shared), first a.smem_entries entries: {skey, meta}, {rem, due}
  uint4 *gtab;             // overflow part (and save area) in global memory, indexed by the same entry index
  const int lane, gl, gshift;   // warp lane, tile lane, first warp lane of the tile
  bool alive;              // the tile holds an environment
  uint32_t env_l;          // its index in the handle's arrays
  uint32_t env_g;          // global env id (Philox counter word)
  // tile-uniform
  int t, epoch, cfg, algo; uint32_t status, n_sys, cfg_sizes;
  uint32_t h_lo, h_hi;
  long long e_ep, tard_ep, busy_ep;
  int P, U, next_crit, repartitioned;
  uint32_t g_k, g_pending, n_accepted, g_done; unsigned long long g_T;   // g_k/g_T: start of the NEXT batch
  uint32_t g_kbase;                                                      // base candidate index of the CURRENT batch
  int look_valid, look_tick, look_work, look_due; uint32_t look_cls, look_id;
  uint32_t n_trace, i_script;
  float ret_acc, disc;     // discounted return so far and gamma^epoch (reading #32)
  // per lane
  uint32_t util_acc;       // tile lane u < 8: seconds spent with u compute units busy
  uint32_t cntA, cntB;     // counters of the current record span (see C_*)
  int g_tick, g_work, g_due; uint32_t g_cls;                             // this lane's candidate of the current batch
  int sl_size, sl_down, sl_upat, sl_pos, sl_rank;                        // slice starting at slot `gl` (gl < 7)
  int rj_rem, rj_due, rj_ctime; uint32_t rj_id, rj_v;                    // job running on it (valid when sl_pos >= 0)

  __device__ __forceinline__ Env(const SimArgs &a_, const HotTables &h_, uint32_t *ws_, uint2 *skm_, uint2 *srd_, int lane_)
      : a(a_), hot(h_), ws(ws_), skm(skm_), srd(srd_), lane(lane_), gl(lane_ & (G - 1)), gshift(lane_ & ~(G - 1)) {}

  // ------------------------------------------------------------------ job table access
  __device__ __forceinline__ uint2 ld_km(uint32_t i) const {
    return i < a.smem_entries ? skm[i] : *reinterpret_cast<const uint2 *>(&gtab[i]);
  }
  __device__ __forceinline__ uint2 ld_rd(uint32_t i) const {
    return i < a.smem_entries ? srd[i] : *(reinterpret_cast<const uint2 *>(&gtab[i]) + 1);
  }
  __device__ __forceinline__ void st_entry(uint32_t i, uint2 km, uint2 rd) {
    if (i < a.smem_entries) { skm[i] = km; srd[i] = rd; } else gtab[i] = make_uint4(km.x, km.y, rd.x, rd.y);
  }
  // word w of entry i: 0 skey, 1 meta, 2 rem, 3 due
  __device__ __forceinline__ uint32_t *entry_word(uint32_t i, int w) {
    if (i < a.smem_entries) return reinterpret_cast<uint32_t *>(w < 2 ? &skm[i] : &srd[i]) + (w & 1);
    return reinterpret_cast<uint32_t *>(&gtab[i]) + w;
  }

  template <int C>
  __device__ __forceinline__ void count(uint32_t n) {
    if constexpr (C < G) cntA += (gl == C) ? n : 0u; else cntB += (gl == C - G) ? n : 0u;
  }
  template <int C>
  __device__ __forceinline__ void count_max(uint32_t v) {
    if constexpr (C < G) { if (gl == C) cntA = max(cntA, v); } else { if (gl == C - G) cntB = max(cntB, v); }
  }
  __device__ __forceinline__ uint32_t counter(int c) const {            // tile-uniform value of counter c (all lanes call)
    return c < G ? T::tshfl(cntA, c) : T::tshfl(cntB, c - G);
  }

  // ------------------------------------------------------------------ trace
  __device__ __forceinline__ void fnv(uint32_t &lo_, uint32_t &hi_, uint32_t w) const {
    // h = (h ^ w) * 0x100000001b3  (64-bit) with 32-bit pieces: h * (2^40 + 0x1b3)
    uint32_t lo = lo_ ^ w, hi = hi_;
    unsigned long long p = (unsigned long long)lo * 0x1b3u;
    lo_ = (uint32_t)p;
    hi_ = (uint32_t)(p >> 32) + hi * 0x1b3u + (lo << 8);
  }
  // every lane executes; the tile's state changes only where pred holds (pred is tile-uniform)
  __device__ __forceinline__ void emit(bool pred, int type, int slot, uint32_t aux, uint32_t job, int value) {
    uint32_t w1 = (uint32_t)type | ((uint32_t)(slot & 0xFF) << 8) | ((aux & 0xFFFFu) << 16);
    uint32_t lo = h_lo, hi = h_hi;
    fnv(lo, hi, (uint32_t)t); fnv(lo, hi, w1); fnv(lo, hi, job); fnv(lo, hi, (uint32_t)value);
    if (pred) { h_lo = lo; h_hi = hi; }
    if (TRACE) {
      if (pred && a.trace && gl == 0 && n_trace < a.trace_cap)
        reinterpret_cast<uint4 *>(a.trace)[n_trace] = make_uint4((uint32_t)t, w1, job, (uint32_t)value);
      if (pred) n_trace++;
    }
    count<C_EVENTS>(pred ? 1u : 0u);
  }

  // ------------------------------------------------------------------ model
  __device__ __forceinline__ int size_at(int p) const { return (cfg_sizes >> (4 * (p & 7))) & 15; }
  __device__ __forceinline__ const uint4 &speed_of(uint32_t cls, int size) const {
    return size == MIG_SIZE_NOMIG ? hot.speed_nomig[cls] : hot.speed[cls * 5 + sidx_of(size)];
  }
  __device__ __forceinline__ int rd(int rem, uint32_t cls, int size) const { return rd_magic(rem, speed_of(cls, size)); }

  // remaining duration against the configuration: fastest slice (LLF) or floor of the mean over all
  // slices of cfg, up or down (LALF; also the state vector's "average duration", L210).  Per-lane loop.
  __device__ __forceinline__ int rd_cfg(int rem, uint32_t cls, bool mean) const {
    int best = MIG_INF, sum = 0, n = 0;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) {
      int g = size_at(p);
      if (g) { int r = rd(rem, cls, g); best = min(best, r); sum += r; ++n; }
    }
    return mean ? sum / n : best;
  }
  __device__ __forceinline__ bool is_lax() const { return (algo & ~1) == MIG_ALGO_LLF; }      // LLF or LALF
  __device__ __forceinline__ int skey_of(int due, int rem, uint32_t cls) const {
    if (!is_lax()) return due;                                  // EDF: deadline
    return due - rd_cfg(rem, cls, algo == MIG_ALGO_LALF);                 // laxity + t (t is common to all jobs)
  }

  __device__ __forceinline__ void update_power(bool pred) {
    bool busy = sl_pos >= 0;
    int c = sl_size ? (busy ? hot.p_busy[sl_size] : hot.p_idle[sl_size]) : 0;
    int u = busy ? tile_units_of(sl_size) : 0;
    int Un = T::tadd(u);
    int Pn = T::tadd(c) + hot.curve[Un & 7];
    if (pred) { U = Un; P = Pn; }
  }

  // rank of this lane's slice among the slices of cfg in (size, slot) order: the tie rule of reading #4 as 3 bits
  __device__ __forceinline__ void compute_rank() {
    int r = 0;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) {
      int g = size_at(p);
      if (g && (g < sl_size || (g == sl_size && p < gl))) ++r;
    }
    sl_rank = r;
  }

  // ------------------------------------------------------------------ arrival generator (R2-R5)
  __device__ __forceinline__ uint32_t neglog2_q24(uint32_t w) const {
    uint32_t m = w | 1u;
    int lz = __clz((int)m);
    uint32_t y = m << lz;
    uint32_t i = (y >> 23) & 0xFFu, f = (y >> 7) & 0xFFFFu;
    uint32_t T0 = __ldg(&a.tab->logT[i]), T1 = __ldg(&a.tab->logT[i + 1]);
    uint32_t L = T0 + (uint32_t)(((unsigned long long)(T1 - T0) * f) >> 16);
    return ((uint32_t)(1 + lz) << 24) - L;
  }

  // generate the batch of G candidates g_k .. g_k+G-1 starting from cumulative time g_T (Q16 seconds); tiles with pred advance
  __device__ __forceinline__ void gen_batch(bool pred) {
    const DevTables *tb = a.tab;
    const uint32_t kbase = g_k; const unsigned long long Tbase = g_T;
    uint32_t k = kbase + (uint32_t)gl;
    uint4 w = philox4x32_10(k, 0u, env_g, a.episode, a.k0, a.k1);            // stream 0: gap, accept, class, slack
    unsigned long long gap = ((unsigned long long)neglog2_q24(w.x) * a.gap_scale) >> 24;
#pragma unroll
    for (int d = 1; d < G; d <<= 1) {                                         // inclusive prefix sum, 64-bit integer
      unsigned long long o = __shfl_up_sync(MIG_FULL, gap, d, G);
      if (gl >= d) gap += o;
    }
    unsigned long long Tc = Tbase + gap;
    unsigned long long tick = Tc >> 16;
    bool in_day = tick < (unsigned long long)a.day_s;                         // arrivals stop at the end of the day
    bool acc = false;
    if (pred && in_day) acc = w.y <= __ldg(&tb->thr[(uint32_t)tick / 60u]);   // Lewis-Shedler thinning
    uint32_t pend = T::tballot(acc, gshift);
    uint32_t dead = T::tballot(pred && !in_day, gshift);
    unsigned long long Tlast = T::tshfl(Tc, G - 1);
    if (pred) {
      g_pending = pend; g_kbase = kbase;
      if (gl == 0) { ws[WS_TBASE] = (uint32_t)Tbase; ws[WS_TBASE + 1] = (uint32_t)(Tbase >> 32); }
      if (dead) g_done = 1;
      else { g_k = kbase + (uint32_t)G; g_T = Tlast; }
    }
    if (acc) {                                                                // job attributes of the accepted ones (per lane)
      uint32_t c = 0;
      for (uint32_t i = 0; i + 1 < a.n_classes; ++i) c += (w.z > __ldg(&tb->class_cum[i])) ? 1u : 0u;
      uint4 wd = philox4x32_10(k, 1u, env_g, a.episode, a.k0, a.k1);          // stream 1: duration
      uint32_t qi = wd.x >> 26, f = (wd.x >> 16) & 0x3FFu;
      int q0 = __ldg(&tb->dur7_q[c * 65 + qi]), q1 = __ldg(&tb->dur7_q[c * 65 + qi + 1]);
      int dur7 = q0 + (int)(((long long)(q1 - q0) * (long long)f) >> 10);
      uint32_t slack = __ldg(&tb->slack_lo[c]) + __umulhi(w.w, __ldg(&tb->slack_span[c]));
      unsigned long long rel = ((unsigned long long)(uint32_t)dur7 * slack) >> 10;
      if (rel < 1) rel = 1;
      g_tick = (int)tick; g_cls = c;
      g_work = (int)((uint32_t)dur7 * hot.speed[c * 5 + 4].x);
      g_due = (int)((long long)tick + (long long)rel);
    }
  }

  // tiles with pred: advance the look-ahead to the next accepted arrival (or none)
  __device__ __forceinline__ void gen_next(bool pred) {
    if (pred) look_valid = 0;
    if (a.script) {                                                           // scripted arrivals (tests), kernel-uniform branch
      if (pred && i_script < a.n_script) {
        mig_job_t s = a.script[i_script];
        look_valid = 1; look_tick = s.arr; look_cls = s.cls; look_due = s.due;
        look_work = (int)((uint32_t)s.dur7 * hot.speed[s.cls * 5 + 4].x);
        look_id = i_script; n_accepted++; i_script++;
      }
      return;
    }
    const uint32_t limit = a.job_limit ? min(a.job_limit, MIG_MAX_JOBS) : MIG_MAX_JOBS;
    const bool need = pred && n_accepted < limit;
    for (;;) {
      bool more = need && !g_pending && !g_done;
      if (!MIG_ANY(more)) break;
      gen_batch(more);
    }
    const bool take = need && g_pending != 0u;
    int l = __ffs((int)g_pending) - 1;
    int tk = T::tshfl(g_tick, l), wk = T::tshfl(g_work, l), du = T::tshfl(g_due, l);
    uint32_t cl = T::tshfl(g_cls, l);
    if (take) {
      g_pending &= g_pending - 1;
      look_tick = tk; look_cls = cl; look_work = wk; look_due = du;
      look_id = n_accepted++;
      look_valid = 1;
    }
  }

  // ------------------------------------------------------------------ reschedule
  // critical-laxity events (LLF / LALF): earliest t_crit = skey - theta > t over waiting jobs
  __device__ __forceinline__ void compute_next_crit(bool go) {
    const bool lax = go && is_lax();
    if (!MIG_ANY(lax)) { if (go) next_crit = MIG_INF; return; }
    int best = MIG_INF;
    if (lax)
      for (uint32_t i = gl; i < n_sys; i += G) {
        uint2 e = ld_km(i);
        int tc = (int)e.x - a.theta;
        bool waiting = ((e.y >> 28) & 7u) == 0u;
        if (waiting && ((e.y >> 24) & 15u) < a.crit_max && tc > t) best = min(best, tc);
      }
    best = T::tmin(best);
    if (go) next_crit = best;
  }

  // EDF-SS with RESTRICTED preemption (reading #26).  Running jobs keep their slices; the
  // waiting jobs are visited in (due, id) order (one tile argmin per visit, "beyond the previous one"): (a) slowest FREE
  // slice on which the job is on time, else (b) slowest OCCUPIED slice on which it is on time among those whose job has
  // a later (due, id): that job is preempted and waits again (it is visited later in the same pass), else (c) fastest
  // free slice, else (d) it waits.  The visit stops when nothing is free and no running job has a later deadline.
  __device__ __forceinline__ void reschedule_restricted(bool go) {
    int pk = (int)0x80000000; uint32_t pid = 0;
    bool open = go;
    for (;;) {
      const bool up = sl_size != 0 && !sl_down;
      const bool any_free = T::tballot(open && up && sl_pos < 0, gshift) != 0u;
      const int max_due = T::tmax((up && sl_pos >= 0) ? rj_due : (int)0x80000000);
      int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu; int bi = -1;
      if (open)
        for (uint32_t i = gl; i < n_sys; i += G) {
          uint2 e = ld_km(i);
          int key = (int)e.x; uint32_t id = e.y & kIdMask;
          bool waiting = ((e.y >> 28) & 7u) == 0u;
          bool beyond = key > pk || (key == pk && id > pid);
          bool better = key < bk || (key == bk && id < bid);
          if (waiting && beyond && better) { bk = key; bid = id; bi = (int)i; }
        }
      const int mk = T::tmin(bk);
      bool cand = bi >= 0 && bk == mk;
      uint32_t cm = T::tballot(cand, gshift);
      if (MIG_ANY((cm & (cm - 1)) != 0u)) {                             // equal deadlines on several lanes: lowest id first
        uint32_t mid = T::tminu(cand ? bid : 0xFFFFFFFFu);
        cm = T::tballot(cand && bid == mid, gshift);
      }
      open = open && cm != 0u && (any_free || mk <= max_due);           // (a deadline equal to max_due may still win on id)
      if (!MIG_ANY(open)) break;
      const int wl = __ffs((int)cm) - 1;
      const uint32_t b = (uint32_t)T::tshfl(bi, wl);
      uint2 km = make_uint2(0u, 0u), rdv = make_uint2(1u, 0u);
      if (open) { km = ld_km(b); rdv = ld_rd(b); }
      const uint32_t cls = (km.y >> 20) & 15u, id = km.y & kIdMask;
      const int rem = (int)rdv.x, due = (int)rdv.y;
      int r = MIG_INF >> 3;
      if (open && up) r = rd_magic(rem, speed_of(cls, sl_size));
      const bool on_time = r <= due - t;
      const bool is_free = open && up && sl_pos < 0;
      const bool later = open && up && sl_pos >= 0 && (rj_due > due || (rj_due == due && rj_id > id));
      const int ssf = (is_free && on_time) ? ((r << 3) | (7 - sl_rank)) : -1;
      const int sso = (later && on_time) ? ((r << 3) | (7 - sl_rank)) : -1;
      const int fsf = is_free ? ((r << 3) | sl_rank) : MIG_INF;
      const int ssfb = T::tmax(ssf), ssob = T::tmax(sso), fsfb = T::tmin(fsf);
      const int mode = ssfb >= 0 ? 0 : (ssob >= 0 ? 1 : (fsfb != MIG_INF ? 2 : 3));
      const bool mine = mode == 0 ? (ssf >= 0 && ssf == ssfb) : (mode == 1 ? (sso >= 0 && sso == ssob) : (mode == 2 && fsf == fsfb));
      const int s = __ffs((int)T::tballot(open && mine, gshift)) - 1;
      if (open) { pk = mk; pid = id; }
      const bool ev = open && mode == 1, st = open && mode != 3;
      const uint32_t vid = T::tshfl(rj_id, s & (G - 1)); const int vrem = T::tshfl(rj_rem, s & (G - 1));
      emit(ev, MIG_EV_PREEMPT, s, (uint32_t)size_at(s), vid, vrem);
      count<C_PREEMPT>(ev ? 1u : 0u);
      if (ev && gl == s) *entry_word((uint32_t)sl_pos, 1) &= ~(7u << 28);          // the evicted job waits again
      __syncwarp();
      emit(st, MIG_EV_START, s, (uint32_t)size_at(s), id, rem);
      count<C_START>(st ? 1u : 0u);
      if (st && gl == s) {
        *entry_word(b, 1) = (km.y & ~(7u << 28)) | ((uint32_t)(s + 1) << 28);
        sl_pos = (int)b; rj_id = id; rj_rem = rem; rj_due = due;
        rj_v = speed_of(cls, sl_size).x;
        rj_ctime = t + r;
      }
      __syncwarp();
    }
    update_power(go);
    if (go) next_crit = MIG_INF;
  }

  // tiles with go re-evaluate every job in the system; the others only keep the warp's instruction stream company
  __device__ __forceinline__ void reschedule(bool go) {
    if (MIG_ANY(go && algo == MIG_ALGO_EDF_SS_R)) {          // (environments of a warp may run different algorithms)
      reschedule_restricted(go && algo == MIG_ALGO_EDF_SS_R);
      go = go && algo != MIG_ALGO_EDF_SS_R;
      if (!MIG_ANY(go)) return;
    }
    const bool busy = sl_pos >= 0;
    if (MIG_ANY(go && is_lax())) {   // the keys of running jobs move with their remaining work
      if (go && is_lax() && busy)
        *entry_word((uint32_t)sl_pos, 0) = (uint32_t)skey_of(rj_due, rj_rem, (ld_km((uint32_t)sl_pos).y >> 20) & 15u);
      __syncwarp();
    }
    uint32_t avail = T::tballot(go && sl_size != 0 && !sl_down, gshift) & 0x7Fu;   // every UP slice, occupied or not
    int K = 0;
    int pk = (int)0x80000000; uint32_t pid = 0;      // (key, id) of the previous pick: the next one is the smallest beyond it
    // rank lane r (< K) remembers the r-th job in priority order
    int asg_slot = -1, asg_old1 = 0, asg_rem = 0; uint32_t asg_id = 0, asg_pos = 0, asg_meta = 0;
    // slice lane p remembers what it will run
    int new_pos = -1, new_rem = 0, new_due = 0, new_r = 0; uint32_t new_id = 0, new_cls = 0;
    for (;;) {
      const bool act = avail != 0u && (uint32_t)K < n_sys;
      if (!MIG_ANY(act)) break;
      // --- next job in (key, id) order: tile argmin over the entries beyond the previous pick (ties -> lower id, reading #5)
      int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu; int bi = -1;
      if (act)
        for (uint32_t i = gl; i < n_sys; i += G) {
          uint2 e = ld_km(i);
          int key = (int)e.x; uint32_t id = e.y & kIdMask;
          bool beyond = key > pk || (key == pk && id > pid);
          bool better = key < bk || (key == bk && id < bid);
          if (beyond && better) { bk = key; bid = id; bi = (int)i; }
        }
      const int mk = T::tmin(bk);
      bool cand = bi >= 0 && bk == mk;
      uint32_t cm = T::tballot(cand, gshift);
      if (MIG_ANY((cm & (cm - 1)) != 0u)) {                             // equal keys on several lanes: lowest id wins
        uint32_t mid = T::tminu(cand ? bid : 0xFFFFFFFFu);
        cm = T::tballot(cand && bid == mid, gshift);
      }
      const int wl = __ffs((int)cm) - 1;
      const uint32_t b = (uint32_t)T::tshfl(bi, wl);
      uint2 km = make_uint2(0u, 0u), rdv = make_uint2(1u, 0u);
      if (act) { km = ld_km(b); rdv = ld_rd(b); }               // broadcast: {skey, meta}, {rem, due}
      const uint32_t cls = (km.y >> 20) & 15u;
      // --- slice choice by the slice lanes: one composite key per rule, (r, rank) unique per lane
      const bool mine = act && ((avail >> gl) & 1u);
      int r = MIG_INF >> 3;
      if (mine) r = rd_magic((int)rdv.x, speed_of(cls, sl_size));
      const int fs = mine ? ((r << 3) | sl_rank) : MIG_INF;                                    // fastest; ties -> smaller size, lower slot (reading #4)
      const int ss = (mine && r <= (int)rdv.y - t) ? ((r << 3) | (7 - sl_rank)) : -1;          // slowest that meets the deadline; same ties
      const int fsb = T::tmin(fs), ssb = T::tmax(ss);
      const bool use_ss = algo == MIG_ALGO_EDF_SS && ssb >= 0;
      const uint32_t pick = T::tballot(mine && (use_ss ? ss == ssb : fs == fsb), gshift);
      const int s = __ffs((int)pick) - 1;
      if (act) {
        avail &= ~(1u << s);
        pk = mk; pid = km.y & kIdMask;
        if (gl == s) { new_pos = (int)b; new_rem = (int)rdv.x; new_due = (int)rdv.y; new_id = km.y & kIdMask; new_cls = cls; new_r = r; }
        if (gl == K) { asg_slot = s; asg_old1 = (int)((km.y >> 28) & 7u); asg_rem = (int)rdv.x; asg_id = km.y & kIdMask; asg_pos = b; asg_meta = km.y; }
        ++K;
      }
    }
    // --- diff against the previous assignment: PREEMPT ascending old slot, START in priority order
    const bool pre = go && busy && new_pos != sl_pos;
    uint32_t pm = T::tballot(pre, gshift);
    count<C_PREEMPT>(__popc(pm));
    while (MIG_ANY(pm != 0u)) {
      int p = __ffs((int)pm) - 1;
      uint32_t id = T::tshfl(rj_id, p); int rem = T::tshfl(rj_rem, p);
      emit(pm != 0u, MIG_EV_PREEMPT, p, (uint32_t)size_at(p), id, rem);
      pm &= pm - 1;
    }
    const bool st = go && gl < K && asg_slot + 1 != asg_old1;
    uint32_t sm = T::tballot(st, gshift);
    count<C_START>(__popc(sm));
    while (MIG_ANY(sm != 0u)) {
      int r_ = __ffs((int)sm) - 1;
      int s = T::tshfl(asg_slot, r_);
      uint32_t id = T::tshfl(asg_id, r_); int rem = T::tshfl(asg_rem, r_);
      emit(sm != 0u, MIG_EV_START, s, (uint32_t)size_at(s), id, rem);
      sm &= sm - 1;
    }
    // --- commit: slot field of the entries, then the slice lanes adopt their jobs
    if (pre) *entry_word((uint32_t)sl_pos, 1) &= ~(7u << 28);
    __syncwarp();
    if (st) *entry_word(asg_pos, 1) = (asg_meta & ~(7u << 28)) | ((uint32_t)(asg_slot + 1) << 28);
    __syncwarp();
    if (go && new_pos != sl_pos) {
      sl_pos = new_pos;
      if (new_pos >= 0) {
        rj_id = new_id; rj_rem = new_rem; rj_due = new_due;
        rj_v = speed_of(new_cls, sl_size).x;
        rj_ctime = t + new_r;
      }
    }
    update_power(go);
    compute_next_crit(go);
  }

  // tiles with pred remove entry `pos` (swap with the last); slice lanes tracking the last entry follow it
  __device__ __forceinline__ void remove_entry(bool pred, uint32_t pos) {
    const uint32_t last = n_sys - 1;
    const bool mv = pred && pos != last;
    uint2 km = make_uint2(0u, 0u), rdv = km;
    if (mv && gl == 0) { km = ld_km(last); rdv = ld_rd(last); }
    __syncwarp();
    if (mv && gl == 0) st_entry(pos, km, rdv);
    if (mv && sl_pos == (int)last) sl_pos = (int)pos;
    if (pred) n_sys = last;
    __syncwarp();
  }

  // ------------------------------------------------------------------ event loop
  // all tiles of the warp advance to t_end (the epoch end, or the drain horizon) in lockstep, one event time per iteration
  __device__ __forceinline__ void run_until(int t_end, bool drain) {
    bool running = alive && !(drain && n_sys == 0);           // drain: energy stops at the last completion (reading #12)
    while (MIG_ANY(running)) {
      // 2. next event time
      int cand = MIG_INF;
      if (sl_pos >= 0) cand = rj_ctime;
      if (sl_size && sl_down) cand = min(cand, sl_upat);
      int tn = min(T::tmin(cand), t_end);
      if (look_valid) tn = min(tn, look_tick);
      tn = min(tn, next_crit);
      const int dt = running ? tn - t : 0;
      e_ep += (long long)P * dt;
      busy_ep += (long long)U * dt;
      if (a.util_hist && gl == U) util_acc += (uint32_t)dt;     // time at this utilisation level (Fig. 6)
      if (sl_pos >= 0 && dt) { rj_rem -= dt * (int)rj_v; *entry_word((uint32_t)sl_pos, 2) = (uint32_t)rj_rem; }
      t += dt;
      __syncwarp();
      // 3. same-tick order (reading #10): completions, slice-ups, arrivals, critical laxity, then ONE reschedule
      bool happened = false;
      uint32_t cm = T::tballot(running && sl_pos >= 0 && rj_rem <= 0, gshift);
      bool job_event = cm != 0u;                                  // a job completed or arrived at this tick
      while (MIG_ANY(cm != 0u)) {                                   // (i) completions, ascending slot
        const bool has = cm != 0u;
        int p = __ffs((int)cm) - 1;
        int due = T::tshfl(rj_due, p);
        uint32_t pos = (uint32_t)T::tshfl(sl_pos, p);
        uint32_t id = T::tshfl(rj_id, p);
        int tard = max(t - due, 0);                           // l_j = max(c_j - d_j, 0)
        emit(has, MIG_EV_COMPLETE, p, (uint32_t)size_at(p), id, tard);
        if (has) tard_ep += tard;
        count<C_COMPLETED>(has ? 1u : 0u); count<C_TARDY>(has && tard > 0 ? 1u : 0u);
        if (has && gl == p) sl_pos = -1;
        remove_entry(has, pos);
        happened |= has;
        cm &= cm - 1;
      }
      uint32_t um = T::tballot(running && sl_size && sl_down && sl_upat == t, gshift);
      while (MIG_ANY(um != 0u)) {                                   // (ii) slices coming up
        const bool has = um != 0u;
        int p = __ffs((int)um) - 1;
        emit(has, MIG_EV_SLICE_UP, p, (uint32_t)size_at(p), MIG_NOJOB, 0);
        if (has && gl == p) sl_down = 0;
        happened |= has;
        um &= um - 1;
      }
      const uint32_t n_before = n_sys;
      for (;;) {                                              // (iii) arrivals, candidate order
        const bool arr = running && look_valid && look_tick == t;
        if (!MIG_ANY(arr)) break;
        const bool drop = arr && n_sys == a.cap;              // queue cap (BASELINE C3/C5)
        const bool ins = arr && !drop;
        count<C_ARRIVED>(arr ? 1u : 0u); count<C_DROPPED>(drop ? 1u : 0u);
        if (ins) {
          int sk = skey_of(look_due, look_work, look_cls);
          if (gl == 0) st_entry(n_sys, make_uint2((uint32_t)sk, look_id | (look_cls << 20)), make_uint2((uint32_t)look_work, (uint32_t)look_due));
          n_sys++;
        }
        emit(arr, drop ? MIG_EV_DROP : MIG_EV_ARRIVE, 0xFF, look_cls, look_id, look_due);
        count_max<C_SYSMAX>(ins ? n_sys : 0u);
        happened |= arr; job_event |= arr;
        gen_next(arr);
      }
      __syncwarp();
      if (MIG_ANY(running && next_crit == t)) {               // (iv) critical laxity, ascending id
        bool scan = running && next_crit == t;
        int last_id = -1;
        for (;;) {
          uint32_t bid = 0xFFFFFFFFu; int bi = -1;
          if (scan)
            for (uint32_t i = gl; i < n_before; i += G) {
              uint2 e = ld_km(i);
              uint32_t id = e.y & kIdMask;
              bool q = ((e.y >> 28) & 7u) == 0u && ((e.y >> 24) & 15u) < a.crit_max && (int)e.x - a.theta == t && (int)id > last_id;
              if (q && id < bid) { bid = id; bi = (int)i; }
            }
          uint32_t mid = T::tminu(bid);
          scan = scan && mid != 0xFFFFFFFFu;
          if (!MIG_ANY(scan)) break;
          int wl = __ffs((int)T::tballot(bid == mid, gshift)) - 1;
          uint32_t b = (uint32_t)T::tshfl(bi, wl);
          uint2 km = make_uint2(0u, 0u), rdv = km;
          if (scan) { km = ld_km(b); rdv = ld_rd(b); }
          uint32_t cc = ((km.y >> 24) & 15u) + 1u;
          __syncwarp();
          if (scan && gl == 0) *entry_word(b, 1) = (km.y & ~(15u << 24)) | (cc << 24);
          __syncwarp();
          emit(scan, MIG_EV_CRIT, 0xFF, cc, mid, (int)rdv.y);
          count<C_CRIT>(scan ? 1u : 0u);
          if (scan) last_id = (int)mid;
          happened |= scan;
        }
      }
      if (a.ev_decide && !drain) {                            // event-driven decision (reading #27)
        const bool dec = running && job_event;
        uint32_t action = (uint32_t)cfg;
        if (a.policy == MIG_POLICY_BINNED) {                  // the paper's binned 2+2m state (L210); every lane takes part
          if (MIG_ANY(dec)) { const uint32_t bi = binned_index(); if (dec) action = a.bin_table[bi]; }
        } else if (dec) {
          const uint32_t b = n_sys == 0 ? 0u : (n_sys < 8 ? 1u : (n_sys < 64 ? 2u : 3u));
          action = a.table[((size_t)env_l * a.n_epochs + epoch) * 4 + b];
        }
        const bool bad = dec && action >= a.n_configs;
        if (bad) status |= MIG_ST_BAD_ACTION;
        const bool rp = dec && !bad && (int)action != cfg;
        if (MIG_ANY(rp)) { repartition(rp, action); happened = happened && !rp; }   // (it reschedules those tiles)
      }
      if (MIG_ANY(happened)) reschedule(happened);            // (v)
      running = running && t != t_end && !(drain && n_sys == 0);
    }
  }

  // ------------------------------------------------------------------ repartition (readings #13, #14)
  __device__ __forceinline__ void prologue(uint32_t action) {
    repartitioned = 0;
    const bool bad = alive && action >= a.n_configs;
    if (bad) status |= MIG_ST_BAD_ACTION;
    const bool rp = alive && !bad && (int)action != cfg;      // "remain on the current configuration": no cost, no event
    if (!MIG_ANY(rp)) return;
    repartition(rp, action);
  }
  // tiles with rp change to the valid configuration `action` (tile-uniform, != cfg); ends with ONE reschedule of those tiles
  __device__ __forceinline__ void repartition(const bool rp, uint32_t action) {
    const uint32_t newsizes = hot.cfg_pack[action & (MIG_MAX_CONFIGS - 1)];
    const int mynew = gl < kSlots ? (int)((newsizes >> (4 * gl)) & 15u) : 0;
    const bool redo = sl_size != mynew || (a.all_down && (sl_size || mynew));   // the whole GPU goes down (reading #30)
    const bool destroyed = rp && sl_size && redo;
    uint32_t pm = T::tballot(destroyed && sl_pos >= 0, gshift);
    count<C_PREEMPT>(__popc(pm));
    while (MIG_ANY(pm != 0u)) {                               // jobs on destroyed slices go back to waiting
      int p = __ffs((int)pm) - 1;
      uint32_t id = T::tshfl(rj_id, p); int rem = T::tshfl(rj_rem, p);
      emit(pm != 0u, MIG_EV_PREEMPT, p, (uint32_t)size_at(p), id, rem);
      pm &= pm - 1;
    }
    if (destroyed && sl_pos >= 0) { *entry_word((uint32_t)sl_pos, 1) &= ~(7u << 28); sl_pos = -1; }
    if (rp && redo) {                                         // same (start, size) in both rows keeps job and up_at
      sl_size = mynew; sl_pos = -1; sl_down = 0; sl_upat = 0;
      if (mynew && a.downtime_s > 0) { sl_down = 1; sl_upat = t + a.downtime_s; }
    }
    const int old = cfg;
    if (rp) { cfg = (int)action; cfg_sizes = newsizes; e_ep += a.repart_energy; repartitioned = 1; compute_rank(); }
    count<C_REPART>(rp ? 1u : 0u);
    emit(rp, MIG_EV_REPART, 0xFF, ((uint32_t)old << 8) | action, MIG_NOJOB, 0);
    __syncwarp();
    if (rp && is_lax())                           // laxity keys are measured against the configuration
      for (uint32_t i = gl; i < n_sys; i += G) {
        uint2 km = ld_km(i), rdv = ld_rd(i);
        *entry_word(i, 0) = (uint32_t)skey_of((int)rdv.y, (int)rdv.x, (km.y >> 20) & 15u);
      }
    __syncwarp();
    reschedule(rp);
  }

  // ------------------------------------------------------------------ records
  __device__ __forceinline__ void begin_span() {
    e_ep = 0; tard_ep = 0; busy_ep = 0;
    cntA = 0; cntB = 0;
    count_max<C_SYSMAX>(n_sys);
    repartitioned = 0;
  }

  // fold the span into the totals; optionally store the 64-byte record (16 words spread over the tile's lanes)
  __device__ __forceinline__ void close_record(mig_epoch_rec_t *r) {
    __syncwarp();
    uint32_t c[C_COUNT];
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) c[i] = counter(i);
    const uint32_t n_run = __popc(T::tballot(sl_pos >= 0, gshift));
    if (gl == 0) {
#pragma unroll
      for (int i = 0; i < C_COUNT; ++i) ws[WS_CNT + i] = (i == C_SYSMAX) ? max(ws[WS_CNT + i], c[i]) : ws[WS_CNT + i] + c[i];
      unsigned long long *tot = reinterpret_cast<unsigned long long *>(&ws[WS_TOT]);
      tot[0] += (unsigned long long)e_ep; tot[1] += (unsigned long long)tard_ep; tot[2] += (unsigned long long)busy_ep;
    }
    __syncwarp();
    if (!r || !alive) return;
    for (int w = gl; w < 16; w += G) {
      uint32_t v = 0;
      switch (w) {
        case 0: v = (uint32_t)e_ep; break;
        case 1: v = (uint32_t)((unsigned long long)e_ep >> 32); break;
        case 2: v = (uint32_t)tard_ep; break;
        case 3: v = (uint32_t)((unsigned long long)tard_ep >> 32); break;
        case 4: v = h_lo; break;
        case 5: v = h_hi; break;
        case 6: v = (uint32_t)busy_ep; break;
        case 7: v = (uint32_t)t; break;
        case 8: v = c[C_EVENTS]; break;
        case 9: v = (c[C_ARRIVED] & 0xFFFFu) | (c[C_COMPLETED] << 16); break;
        case 10: v = (c[C_DROPPED] & 0xFFFFu) | (c[C_TARDY] << 16); break;
        case 11: v = (c[C_PREEMPT] & 0xFFFFu) | (c[C_START] << 16); break;
        case 12: v = (c[C_CRIT] & 0xFFFFu) | (n_sys << 16); break;
        case 13: v = (uint32_t)cfg | ((uint32_t)repartitioned << 8) | ((status & 0xFFu) << 16) | (n_run << 24); break;
        case 14: v = c[C_SYSMAX]; break;
        default: v = 0; break;
      }
      reinterpret_cast<uint32_t *>(r)[w] = v;
    }
  }

  // word order of mig_totals_t: energy(0,1) tard(2,3) hash(4,5) busy(6,7) n_jobs..n_sys_max(8..17) t_end(18) status(19)
  __device__ __forceinline__ void store_totals(mig_totals_t *o) {
    __syncwarp();
    if (!alive) return;
    for (int w = gl; w < 20; w += G) {
      uint32_t v;
      if (w < 8) v = (w == 4) ? h_lo : (w == 5) ? h_hi : ws[WS_TOT + (w < 4 ? w : w - 2)];
      else if (w < 18) v = ws[WS_CNT + (w - 8)];
      else v = (w == 18) ? (uint32_t)t : status;
      reinterpret_cast<uint32_t *>(o)[w] = v;
    }
  }

  // ------------------------------------------------------------------ state vector
  __device__ __forceinline__ void observe(float *out) {
    uint32_t *st = ws + WS_STAGE;
    __syncwarp();
    for (int w = gl; w < MIG_STATE_DIM; w += G) st[w] = 0u;
    __syncwarp();
    for (uint32_t i = gl; i < n_sys; i += G) {                 // waiting jobs per class
      uint32_t m = ld_km(i).y;
      if (((m >> 28) & 7u) == 0u) atomicAdd(&st[(m >> 20) & 15u], 1u);
    }
    __syncwarp();
    if (gl < 16) st[gl] = __float_as_uint((float)st[gl]);
    if (G < 16 && gl + 8 < 16) st[gl + 8] = __float_as_uint((float)st[gl + 8]);
    const uint32_t n_run = __popc(T::tballot(sl_pos >= 0, gshift));
    if (gl < kSlots) {
      const float occ = sl_down ? 0.5f : (sl_pos >= 0 ? 1.0f : 0.0f);
      for (int q = 0; q < tile_units_of(sl_size); ++q) st[16 + gl + q] = __float_as_uint(occ);        // slots covered by this slice
      st[23 + gl] = __float_as_uint((float)sl_size * 0.125f);
    }
    if (gl == 7 % G) {
      st[30 + (t / 3600) % 24] = __float_as_uint(1.0f);
      st[54] = __float_as_uint((float)(n_sys - n_run) * (1.0f / 64.0f));
      st[55] = __float_as_uint((float)n_run * 0.125f);
      st[62] = __float_as_uint((float)ws[WS_DROPS] * (1.0f / 64.0f));
      st[63] = __float_as_uint(1.0f);
    }
    int pk = (int)0x80000000; uint32_t pid = 0;
#pragma unroll 1
    for (int m = 0; m < 3; ++m) {                               // first m = 3 jobs in (due, id) order
      const bool act = (uint32_t)m < n_sys;
      const uint32_t b = next_by_due(act, pk, pid);
      if (act) {
        uint2 km = ld_km(b), rdv = ld_rd(b);
        int d = max(-32768, min(32767, (int)rdv.y - t));
        int mean = min(rd_cfg((int)rdv.x, (km.y >> 20) & 15u, true), 32767);
        if (gl == 0) { st[56 + m] = __float_as_uint((float)d * (1.0f / 4096.0f)); st[59 + m] = __float_as_uint((float)mean * (1.0f / 4096.0f)); }
      }
    }
    __syncwarp();
    if (alive)
      for (int w = gl; w < MIG_STATE_DIM; w += G) out[w] = __uint_as_float(st[w]);
    __syncwarp();
  }
  // tiles with act: entry index of the job that follows (pk, pid) in (due, id) order over all jobs in system (running and
  // waiting); advances (pk, pid).  One tile argmin; every lane of the warp executes it.
  __device__ __forceinline__ uint32_t next_by_due(bool act, int &pk, uint32_t &pid) {
    int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu; int bi = -1;
    if (act)
      for (uint32_t i = gl; i < n_sys; i += G) {
        int due = (int)ld_rd(i).y; uint32_t id = ld_km(i).y & kIdMask;
        bool beyond = due > pk || (due == pk && id > pid);
        bool better = due < bk || (due == bk && id < bid);
        if (beyond && better) { bk = due; bid = id; bi = (int)i; }
      }
    const int mk = T::tmin(bk);
    const uint32_t mid = T::tminu((bi >= 0 && bk == mk) ? bid : 0xFFFFFFFFu);
    const int wl = __ffs((int)T::tballot(bi >= 0 && bk == mk && bid == mid, gshift)) - 1;
    const uint32_t b = (uint32_t)T::tshfl(bi, wl);
    if (act) { pk = mk; pid = mid; }
    return b;
  }

  // ------------------------------------------------------------------ binned state (reading #31)
  // index of the present state in the BINNED policy's table: configuration, time bin, and for each of the first m = 3 jobs
  // in (due, id) order the code 0 (no such job) or 1 + dbin * n_abins + abin of its deadline (due - t) and its mean
  // remaining duration over the slices of the configuration.  Tile-uniform; every lane of the warp executes it.
  static __device__ __forceinline__ uint32_t bin_of(int v, const int32_t *edges, uint32_t n_bins) {
    uint32_t b = 0;
    while (b + 1u < n_bins && v >= __ldg(&edges[b])) ++b;
    return b;
  }
  __device__ __forceinline__ uint32_t binned_index() {
    const uint32_t B = 1u + a.n_dbins * a.n_abins;
    const uint32_t tc = (uint32_t)min(t, a.day_s - 1);
    uint32_t idx = (uint32_t)cfg * a.n_tbins + (tc * a.n_tbins) / (uint32_t)a.day_s;
    int pk = (int)0x80000000; uint32_t pid = 0;
    __syncwarp();
#pragma unroll 1
    for (uint32_t m = 0; m < 3u; ++m) {
      const bool act = m < n_sys;
      const uint32_t b = next_by_due(act, pk, pid);
      uint32_t code = 0;
      if (act) {
        const uint2 km = ld_km(b), rdv = ld_rd(b);
        const uint32_t db = bin_of((int)rdv.y - t, a.tab->dbin_edges, a.n_dbins);
        const uint32_t ab = bin_of(rd_cfg((int)rdv.x, (km.y >> 20) & 15u, true), a.tab->abin_edges, a.n_abins);
        code = 1u + db * a.n_abins + ab;
      }
      idx = idx * B + code;
    }
    return idx;
  }

  // ------------------------------------------------------------------ init / load / save
  __device__ __forceinline__ void set_config(int c) {
    cfg = c; cfg_sizes = hot.cfg_pack[c];
    sl_size = gl < kSlots ? size_at(gl) : 0;
    sl_down = 0; sl_upat = 0; sl_pos = -1;
    compute_rank();
  }

  __device__ __forceinline__ void clear_lane_state() {
    rj_rem = 0; rj_due = 0; rj_ctime = 0; rj_id = 0; rj_v = 0;
    g_tick = 0; g_work = 0; g_due = 0; g_cls = 0;
    cntA = 0; cntB = 0;
  }

  __device__ __forceinline__ void init(uint32_t env_local) {
    algo = a.algo[env_local]; t = 0; epoch = 0; status = 0; n_sys = 0;
    if (algo > MIG_ALGO_EDF_SS_R) { algo = MIG_ALGO_EDF_FS; status |= MIG_ST_BAD_ALGO; }   // reading #28
    h_lo = 0x84222325u; h_hi = 0xcbf29ce4u;                   // FNV-1a-64 offset basis
    uint32_t c0 = a.cfg0[env_local];
    if (c0 >= a.n_configs) { c0 = 0; status |= MIG_ST_BAD_ACTION; }
    set_config((int)c0);
    clear_lane_state();
    g_k = 0; g_T = 0; g_pending = 0; n_accepted = 0; g_done = 0; g_kbase = 0;
    look_valid = 0; look_tick = 0; look_work = 0; look_due = 0; look_cls = 0; look_id = 0;
    next_crit = MIG_INF; n_trace = 0; i_script = 0; P = 0; U = 0;
    util_acc = 0; ret_acc = 0.0f; disc = 1.0f;
    __syncwarp();
    for (int w = gl; w < WS_WORDS; w += G) ws[w] = 0;
    __syncwarp();
    begin_span();
    update_power(true);
    gen_next(alive);
  }

  __device__ __forceinline__ void save(uint32_t env_local) {
    uint32_t *st = ws + WS_STAGE;
    __syncwarp();
    if (gl == 0) {
      st[H_T] = (uint32_t)t;
      st[H_PK] = (uint32_t)epoch | ((uint32_t)cfg << 8) | ((uint32_t)algo << 16) | (status << 24);
      st[H_NSYS] = n_sys; st[H_HLO] = h_lo; st[H_HHI] = h_hi;
      st[H_GKBASE] = g_kbase; st[H_TBASE_LO] = ws[WS_TBASE]; st[H_TBASE_HI] = ws[WS_TBASE + 1];
      st[H_GPENDING] = g_pending; st[H_NACC] = n_accepted; st[H_GDONE] = g_done; st[H_ISCRIPT] = i_script;
      st[H_DROPS] = ws[WS_DROPS];
#pragma unroll
      for (int i = 0; i < 6; ++i) st[H_TOT + i] = ws[WS_TOT + i];
      st[H_LOOKV] = (uint32_t)look_valid; st[H_LOOKTICK] = (uint32_t)look_tick; st[H_LOOKCLS] = look_cls;
      st[H_LOOKWORK] = (uint32_t)look_work; st[H_LOOKDUE] = (uint32_t)look_due; st[H_LOOKID] = look_id;
      st[H_GK] = g_k; st[H_GT_LO] = (uint32_t)g_T; st[H_GT_HI] = (uint32_t)(g_T >> 32);
      st[H_RET] = __float_as_uint(ret_acc); st[H_DISC] = __float_as_uint(disc);
#pragma unroll
      for (int i = 0; i < C_COUNT; ++i) st[H_CNT + i] = ws[WS_CNT + i];
    }
    if (gl < 8) st[tile_util_word(gl)] = util_acc;
    if (gl < kSlots) {
      st[H_UPAT + gl] = (uint32_t)sl_upat;
      st[H_SLICE + gl] = (uint32_t)sl_size | ((uint32_t)sl_down << 8) | ((uint32_t)(sl_pos + 1) << 16);
    }
    __syncwarp();
    if (alive) {
      uint32_t *h = a.hdr + (size_t)env_local * kHeaderWords;
      for (int w = gl; w < kHeaderWords; w += G) h[w] = st[w];
      const uint32_t ns = min(n_sys, a.smem_entries);
      for (uint32_t i = gl; i < ns; i += G) { uint2 km = skm[i], rdv = srd[i]; gtab[i] = make_uint4(km.x, km.y, rdv.x, rdv.y); }
    }
    __syncwarp();
  }

  __device__ __forceinline__ void load(uint32_t env_local) {
    uint32_t *st = ws + WS_STAGE;
    const uint32_t *h = a.hdr + (size_t)env_local * kHeaderWords;
    __syncwarp();
    for (int w = gl; w < WS_WORDS; w += G) ws[w] = w < kHeaderWords ? h[w] : 0u;
    __syncwarp();
    t = (int)st[H_T];
    const uint32_t pk = st[H_PK];
    epoch = pk & 0xFF; cfg = (pk >> 8) & 0xFF; algo = (pk >> 16) & 0xFF; status = pk >> 24;
    n_sys = st[H_NSYS]; h_lo = st[H_HLO]; h_hi = st[H_HHI];
    const uint32_t kb = st[H_GKBASE], tb_lo = st[H_TBASE_LO], tb_hi = st[H_TBASE_HI], pend = st[H_GPENDING];
    n_accepted = st[H_NACC];
    const uint32_t gd = st[H_GDONE];
    i_script = st[H_ISCRIPT];
    const uint32_t drops = st[H_DROPS];
    uint32_t tot[6], cnt[C_COUNT];
#pragma unroll
    for (int i = 0; i < 6; ++i) tot[i] = st[H_TOT + i];
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) cnt[i] = st[H_CNT + i];
    look_valid = (int)st[H_LOOKV]; look_tick = (int)st[H_LOOKTICK]; look_cls = st[H_LOOKCLS];
    look_work = (int)st[H_LOOKWORK]; look_due = (int)st[H_LOOKDUE]; look_id = st[H_LOOKID];
    const uint32_t gk = st[H_GK];
    ret_acc = __uint_as_float(st[H_RET]); disc = __uint_as_float(st[H_DISC]);
    util_acc = gl < 8 ? st[tile_util_word(gl)] : 0u;
    const unsigned long long gT = (unsigned long long)st[H_GT_LO] | ((unsigned long long)st[H_GT_HI] << 32);
    cfg_sizes = hot.cfg_pack[cfg & (MIG_MAX_CONFIGS - 1)];
    sl_size = 0; sl_down = 0; sl_upat = 0; sl_pos = -1;
    if (gl < kSlots) {
      const uint32_t w1 = st[H_SLICE + gl];
      sl_upat = (int)st[H_UPAT + gl]; sl_size = w1 & 0xFF; sl_down = (w1 >> 8) & 0xFF; sl_pos = (int)(w1 >> 16) - 1;
    }
    compute_rank();
    __syncwarp();
    for (int w = gl; w < kHeaderWords; w += G) st[w] = 0u;     // the staging area becomes scratch again
    __syncwarp();
    if (gl == 0) {
#pragma unroll
      for (int i = 0; i < 6; ++i) ws[WS_TOT + i] = tot[i];
#pragma unroll
      for (int i = 0; i < C_COUNT; ++i) ws[WS_CNT + i] = cnt[i];
      ws[WS_TBASE] = tb_lo; ws[WS_TBASE + 1] = tb_hi; ws[WS_DROPS] = drops;
    }
    const uint32_t ns = min(n_sys, a.smem_entries);
    for (uint32_t i = gl; i < ns; i += G) { uint4 e = gtab[i]; skm[i] = make_uint2(e.x, e.y); srd[i] = make_uint2(e.z, e.w); }
    __syncwarp();
    clear_lane_state();
    g_pending = 0; g_done = 0; g_kbase = kb;
    g_k = kb; g_T = (unsigned long long)tb_lo | ((unsigned long long)tb_hi << 32);
    if (MIG_ANY(pend != 0u)) gen_batch(pend != 0u);           // rebuild the candidates of the batch in flight
    g_k = gk; g_T = gT; g_done = gd; g_pending = pend; g_kbase = kb;
    if (gl == 0) { ws[WS_TBASE] = tb_lo; ws[WS_TBASE + 1] = tb_hi; }
    if (sl_pos >= 0) {                                       // running job: t + ceil(rem / v) never drifts
      uint2 km = ld_km((uint32_t)sl_pos), rdv = ld_rd((uint32_t)sl_pos);
      uint4 sp = speed_of((km.y >> 20) & 15u, sl_size);
      rj_id = km.y & kIdMask; rj_rem = (int)rdv.x; rj_due = (int)rdv.y; rj_v = sp.x;
      rj_ctime = t + rd_magic(rj_rem, sp);
    }
    n_trace = 0; P = 0; U = 0; next_crit = MIG_INF;
    begin_span();
    update_power(true);
    compute_next_crit(true);
  }

  // ------------------------------------------------------------------ one decision epoch
  __device__ __forceinline__ void step(uint32_t env_local, uint32_t action) {
    const int k = epoch;
    begin_span();
    prologue(action);
    run_until((k + 1) * a.epoch_s, false);
    long long dE = e_ep, dT = tard_ep;
    const uint32_t drops = counter(C_DROPPED);
    __syncwarp();
    if (gl == 0) ws[WS_DROPS] = drops;
    close_record(a.recs ? a.recs + (size_t)(k - a.rec_k0) * a.rec_stride + env_local : nullptr);
    if (k == a.n_epochs - 1) {                                // 4. drain (reading #11)
      begin_span();
      run_until(a.t_limit_s, true);
      if (n_sys > 0) status |= MIG_ST_TRUNCATED;
      dE += e_ep; dT += tard_ep;
      close_record(a.drain_rec ? a.drain_rec + env_local : nullptr);
    }
    epoch = k + 1;
    // reward: two fp32 products, one add, negate; no contraction
    const float r = -__fadd_rn(__fmul_rn(a.w_energy, __ll2float_rn(dE)), __fmul_rn(a.w_tardy, __ll2float_rn(dT)));
    if (alive && gl == 0) {
      if (a.energy_out) a.energy_out[env_local] = dE;
      if (a.tard_out) a.tard_out[env_local] = dT;
      if (a.reward_out) a.reward_out[env_local] = r;
    }
    ret_acc = __fmaf_rn(disc, r, ret_acc);                    // discounted return (reading #32)
    disc = __fmul_rn(disc, a.gamma);
  }
};

template <int G, bool TRACE>
__global__ void __launch_bounds__(kWarpsPerCta * 32, 4) sim_kernel(const SimArgs a) {
  constexpr int NG = 32 / G;                                  // environments per warp
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HotTables &hot = *reinterpret_cast<HotTables *>(smem_raw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  {
    const DevTables *tb = a.tab;
    for (int i = threadIdx.x; i < MIG_MAX_CLASSES * 5; i += blockDim.x) hot.speed[i] = tb->speed[i];
    for (int i = threadIdx.x; i < MIG_MAX_CONFIGS; i += blockDim.x) hot.cfg_pack[i] = tb->cfg_pack[i];
    for (int i = threadIdx.x; i < MIG_MAX_CLASSES; i += blockDim.x) hot.speed_nomig[i] = tb->speed_nomig[i];
    if (threadIdx.x < 8) hot.curve[threadIdx.x] = tb->curve[threadIdx.x];
    if (threadIdx.x < 12) { hot.p_idle[threadIdx.x] = tb->p_idle[threadIdx.x]; hot.p_busy[threadIdx.x] = tb->p_busy[threadIdx.x]; }
  }
  __syncthreads();
  const size_t per_tile = tile_smem_bytes(a.smem_entries);
  unsigned char *base = smem_raw + ((sizeof(HotTables) + 127) & ~(size_t)127) + (size_t)(warp * NG + lane / G) * per_tile;
  uint32_t *ws = reinterpret_cast<uint32_t *>(base);
  uint2 *skm = reinterpret_cast<uint2 *>(base + WS_WORDS * 4);
  uint2 *srd = skm + a.smem_entries;
  Env<G, TRACE> e(a, hot, ws, skm, srd, lane);
  for (;;) {
    uint32_t idx = 0;
    if (lane == 0) idx = atomicAdd(a.counter, 1u);
    idx = __shfl_sync(MIG_FULL, idx, 0);
    if (idx * NG >= a.n_envs) break;
    const uint32_t li = idx * NG + (uint32_t)(lane / G);      // index inside this launch's env range
    e.alive = li < a.n_envs;
    const uint32_t env = a.env_first + (e.alive ? li : 0u);   // idle tiles shadow a valid env and never write
    e.env_g = a.env_base + env; e.env_l = env;
    e.gtab = a.tab_override ? a.tab_override : a.jobtab + (size_t)env * a.cap;
    if (a.from_init) e.init(env); else e.load(env);
    for (int s = 0; s < a.n_steps && e.epoch < a.n_epochs; ++s) {
      uint32_t action = (uint32_t)e.cfg;                                            // STATIC: stay
      if (a.policy == MIG_POLICY_TABLE) {                                           // load bucket
        uint32_t b = e.n_sys == 0 ? 0u : (e.n_sys < 8 ? 1u : (e.n_sys < 64 ? 2u : 3u));
        action = a.table[((size_t)env * a.n_epochs + e.epoch) * 4 + b];
      } else if (a.policy == MIG_POLICY_BINNED) {                                   // binned 2+2m state
        action = a.bin_table[e.binned_index()];
      } else if (a.actions) {
        action = a.actions[(size_t)(e.alive ? li : 0u) * a.act_stride_env + (size_t)s * a.act_stride_k];
      }
      e.step(TRACE ? 0u : env, action);
    }
    if (a.state_out) e.observe(a.state_out + (size_t)(TRACE ? 0u : env) * MIG_STATE_DIM);
    if (a.totals) e.store_totals(a.totals + (TRACE ? 0u : env));   // totals so far (hash and t are live values)
    if (a.save) e.save(env);
    if (TRACE && a.trace_n && lane == 0) *a.trace_n = e.n_trace;
    __syncwarp();
  }
}

}  // namespace migsim
