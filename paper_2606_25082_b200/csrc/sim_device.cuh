// sim_device.cuh -- the rollout kernel: ONE WARP PER ENVIRONMENT (north_star (a)).
//
// Each warp simulates one MIG-partitioned GPU through `n_steps` decision epochs, event by event
// (every arrival / completion is a preemption point at which ALL jobs in the system are re-evaluated).
//   * job table {skey, meta, rem, due} (16 B / job) in shared memory (first `smem_entries`), overflow in global;
//   * slice table: lane p < 7 owns the slice that starts at slot p (size, down/up, running job cached in registers);
//   * reschedule = up to 7 warp-argmin passes over the priority key (REDUX + ballot), slice choice by the 7 slice lanes
//     in parallel (one exact magic-number division each), PREEMPT/START diff;
//   * arrivals: counter-based Philox4x32-10, 32 thinning candidates per warp pass (one per lane), gaps prefix-summed
//     in 64-bit fixed point (integer => associative => identical to sequential accumulation);
//   * energy / tardiness in int64, trace hash FNV-1a-64 over every event.
// All readings (tie rules, same-tick order, drain, ...) are DESIGN.md section 3.  No code is shared with oracle/.
#pragma once
#include <cuda_runtime.h>

#include "sim_common.h"

namespace migsim {

#define MIG_FULL 0xffffffffu
#define MIG_INF 0x7fffffff

// counters, lane-indexed: lane 16 + c holds counter c
enum { C_ARRIVED = 0, C_COMPLETED, C_DROPPED, C_TARDY, C_PREEMPT, C_START, C_CRIT, C_EVENTS, C_REPART, C_SYSMAX };   // = word order of mig_totals_t

// per-warp scratch in shared memory (words)
enum { WS_CLS = 0, WS_CNT = 16, WS_TOT = 26 /* 3 x u64 */, WS_TBASE = 32 /* u64 */, WS_DROPS = 34, WS_ISCRIPT = 35,
       WS_WORDS = 64 };

struct HotTables {               // per CTA, shared memory
  uint4 speed[MIG_MAX_CLASSES * 5];
  uint32_t cfg_pack[MIG_MAX_CONFIGS];
  int32_t curve[8], p_idle[8], p_busy[8];
};

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
  // Salmon et al., SC'11: ten rounds of two 32x32->64 multiplies, key bumped by the Weyl constants (R1)
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ int sidx_of(int size) { return size == 7 ? 4 : size - 1; }   // 1,2,3,4,7 -> 0..4

// ceil(rem / v) for 0 < rem, rem + v - 1 < 2^31, by the precomputed magic number of v (exact; see mig_debug_div_magic)
__device__ __forceinline__ int rd_magic(int rem, uint4 sp) {
  uint32_t x = (uint32_t)rem + sp.x - 1u;
  uint32_t q = __umulhi(x, sp.y) >> (sp.z & 31u);
  return (int)(sp.z >= 32u ? x : q);
}

template <bool TRACE>
struct Env {
  // ------------------------------------------------------------------ environment state (registers)
  const SimArgs &a;
  const HotTables &hot;
  uint32_t *ws;            // per-warp scratch (shared)
  uint4 *stab;             // per-warp job table (shared), first a.smem_entries entries
  uint4 *gtab;             // overflow part in global memory, indexed by the same entry index
  const int lane;
  uint32_t env_g;          // global env id (Philox counter word)
  // uniform
  int t, epoch, cfg, algo; uint32_t status, n_sys, cfg_sizes;
  uint32_t h_lo, h_hi;
  long long e_ep, tard_ep, busy_ep;
  int P, U, next_crit, repartitioned;
  uint32_t g_k, g_pending, n_accepted, g_done; unsigned long long g_T;   // g_k/g_T: start of the NEXT batch
  uint32_t g_kbase;                                                      // base candidate index of the CURRENT batch
  int look_valid, look_tick, look_work, look_due; uint32_t look_cls, look_id;
  uint32_t n_trace;
  // per lane
  uint32_t cnt_ep;         // lane 16 + c: counter c of the current record span
  int g_tick, g_work, g_due; uint32_t g_cls;                             // this lane's candidate of the current batch
  int sl_size, sl_down, sl_upat, sl_pos;                                 // slice starting at slot `lane` (lane < 7)
  int rj_rem, rj_due, rj_ctime; uint32_t rj_id, rj_v;                    // job running on it (valid when sl_pos >= 0)

  __device__ __forceinline__ Env(const SimArgs &a_, const HotTables &h_, uint32_t *ws_, uint4 *stab_, int lane_)
      : a(a_), hot(h_), ws(ws_), stab(stab_), lane(lane_) {}

  // ------------------------------------------------------------------ job table access
  __device__ __forceinline__ uint4 ld_entry(uint32_t i) const { return i < a.smem_entries ? stab[i] : gtab[i]; }
  __device__ __forceinline__ void st_entry(uint32_t i, uint4 e) { if (i < a.smem_entries) stab[i] = e; else gtab[i] = e; }
  __device__ __forceinline__ uint2 ld_key(uint32_t i) const {
    return i < a.smem_entries ? *reinterpret_cast<const uint2 *>(&stab[i]) : *reinterpret_cast<const uint2 *>(&gtab[i]);
  }
  __device__ __forceinline__ uint32_t *entry_word(uint32_t i, int w) {
    return (i < a.smem_entries ? reinterpret_cast<uint32_t *>(&stab[i]) : reinterpret_cast<uint32_t *>(&gtab[i])) + w;
  }

  __device__ __forceinline__ void count(int c, uint32_t n = 1) { cnt_ep += (lane == 16 + c) ? n : 0u; }

  // ------------------------------------------------------------------ trace
  __device__ __forceinline__ void fnv(uint32_t w) {
    // h = (h ^ w) * 0x100000001b3  (64-bit) with 32-bit pieces: h * (2^40 + 0x1b3)
    uint32_t lo = h_lo ^ w, hi = h_hi;
    unsigned long long p = (unsigned long long)lo * 0x1b3u;
    h_lo = (uint32_t)p;
    h_hi = (uint32_t)(p >> 32) + hi * 0x1b3u + (lo << 8);
  }
  __device__ __forceinline__ void emit(int type, int slot, uint32_t aux, uint32_t job, int value) {
    uint32_t w1 = (uint32_t)type | ((uint32_t)(slot & 0xFF) << 8) | ((aux & 0xFFFFu) << 16);
    fnv((uint32_t)t); fnv(w1); fnv(job); fnv((uint32_t)value);
    if (TRACE) {
      if (a.trace && lane == 0 && n_trace < a.trace_cap)
        reinterpret_cast<uint4 *>(a.trace)[n_trace] = make_uint4((uint32_t)t, w1, job, (uint32_t)value);
      n_trace++;
    }
    count(C_EVENTS);
  }

  // ------------------------------------------------------------------ model
  __device__ __forceinline__ int size_at(int p) const { return (cfg_sizes >> (4 * p)) & 15; }
  __device__ __forceinline__ int rd(int rem, uint32_t cls, int size) const { return rd_magic(rem, hot.speed[cls * 5 + sidx_of(size)]); }

  // remaining duration against the configuration: fastest slice (LLF) or floor of the mean over all
  // slices of cfg, up or down (LALF; also the state vector's "average duration", L210).  Uniform loop.
  __device__ __forceinline__ int rd_cfg(int rem, uint32_t cls, bool mean) const {
    int best = MIG_INF, sum = 0, n = 0;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) {
      int g = size_at(p);
      if (g) { int r = rd(rem, cls, g); best = min(best, r); sum += r; ++n; }
    }
    return mean ? sum / n : best;
  }
  __device__ __forceinline__ int skey_of(int due, int rem, uint32_t cls) const {
    if (algo < MIG_ALGO_LLF) return due;                                  // EDF: deadline
    return due - rd_cfg(rem, cls, algo == MIG_ALGO_LALF);                 // laxity + t (t is common to all jobs)
  }

  __device__ __forceinline__ void update_power() {
    bool busy = sl_pos >= 0;
    int c = sl_size ? (busy ? hot.p_busy[sl_size] : hot.p_idle[sl_size]) : 0;
    int u = busy ? sl_size : 0;
    U = __reduce_add_sync(MIG_FULL, u);
    P = __reduce_add_sync(MIG_FULL, c) + hot.curve[U];
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

  // generate the batch of 32 candidates kbase .. kbase+31 starting from cumulative time Tbase (Q16 seconds)
  __device__ __forceinline__ void gen_batch(uint32_t kbase, unsigned long long Tbase) {
    const DevTables *tb = a.tab;
    uint32_t k = kbase + (uint32_t)lane;
    uint4 w = philox4x32_10(k, 0u, env_g, a.episode, a.k0, a.k1);            // stream 0: gap, accept, class, slack
    unsigned long long gap = ((unsigned long long)neglog2_q24(w.x) * a.gap_scale) >> 24;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {                                        // inclusive prefix sum, 64-bit integer
      unsigned long long o = __shfl_up_sync(MIG_FULL, gap, d);
      if (lane >= d) gap += o;
    }
    unsigned long long T = Tbase + gap;
    unsigned long long tick = T >> 16;
    bool in_day = tick < (unsigned long long)a.day_s;                         // arrivals stop at the end of the day
    bool acc = false;
    if (in_day) acc = w.y <= __ldg(&tb->thr[(uint32_t)tick / 60u]);           // Lewis-Shedler thinning
    g_pending = __ballot_sync(MIG_FULL, acc);
    uint32_t dead = __ballot_sync(MIG_FULL, !in_day);
    g_kbase = kbase;
    ws[WS_TBASE] = (uint32_t)Tbase; ws[WS_TBASE + 1] = (uint32_t)(Tbase >> 32);
    if (dead) g_done = 1;
    else { g_k = kbase + 32u; g_T = __shfl_sync(MIG_FULL, T, 31); }
    if (g_pending) {                                                          // job attributes of the accepted ones
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

  // advance the look-ahead to the next accepted arrival (or none)
  __device__ __forceinline__ void gen_next() {
    look_valid = 0;
    if (a.script) {
      uint32_t i = ws[WS_ISCRIPT];
      if (i < a.n_script) {
        mig_job_t s = a.script[i];
        look_valid = 1; look_tick = s.arr; look_cls = s.cls; look_due = s.due;
        look_work = (int)((uint32_t)s.dur7 * hot.speed[s.cls * 5 + 4].x);
        look_id = i; n_accepted++;
        __syncwarp();
        ws[WS_ISCRIPT] = i + 1;
        __syncwarp();
      }
      return;
    }
    uint32_t limit = a.job_limit ? min(a.job_limit, MIG_MAX_JOBS) : MIG_MAX_JOBS;
    if (n_accepted >= limit) return;
    while (!g_pending && !g_done) gen_batch(g_k, g_T);
    if (!g_pending) return;
    int l = __ffs((int)g_pending) - 1;
    g_pending &= g_pending - 1;
    look_tick = __shfl_sync(MIG_FULL, g_tick, l);
    look_cls = __shfl_sync(MIG_FULL, g_cls, l);
    look_work = __shfl_sync(MIG_FULL, g_work, l);
    look_due = __shfl_sync(MIG_FULL, g_due, l);
    look_id = n_accepted++;
    look_valid = 1;
  }

  // ------------------------------------------------------------------ reschedule
  // critical-laxity events (LLF / LALF): earliest t_crit = skey - theta > t over waiting jobs
  __device__ __forceinline__ void compute_next_crit() {
    next_crit = MIG_INF;
    if (algo < MIG_ALGO_LLF) return;
    int best = MIG_INF;
    for (uint32_t i = lane; i < n_sys; i += 32) {
      uint2 e = ld_key(i);
      int tc = (int)e.x - a.theta;
      bool waiting = ((e.y >> 28) & 7u) == 0u;
      if (waiting && ((e.y >> 24) & 15u) < a.crit_max && tc > t) best = min(best, tc);
    }
    next_crit = __reduce_min_sync(MIG_FULL, best);
  }

  __device__ __forceinline__ void reschedule() {
    const bool busy = sl_pos >= 0;
    if (algo >= MIG_ALGO_LLF) {                 // the keys of running jobs move with their remaining work
      if (busy) *entry_word((uint32_t)sl_pos, 0) = (uint32_t)skey_of(rj_due, rj_rem, (ld_key((uint32_t)sl_pos).y >> 20) & 15u);
      __syncwarp();
    }
    uint32_t avail = __ballot_sync(MIG_FULL, sl_size != 0 && !sl_down) & 0x7Fu;   // every UP slice, occupied or not
    uint32_t taken = 0;                          // bit j: entry lane + 32 j already placed
    int K = 0;
    // rank lane r (< K) remembers the r-th job in priority order
    int asg_slot = -1, asg_old1 = 0, asg_rem = 0; uint32_t asg_id = 0, asg_pos = 0, asg_meta = 0;
    // slice lane p remembers what it will run
    int new_pos = -1, new_rem = 0, new_due = 0, new_r = 0; uint32_t new_id = 0, new_cls = 0;
    while (avail && (uint32_t)K < n_sys) {
      // --- next job in (key, id) order: warp argmin (ties -> lower id, reading #5)
      int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu; int bi = -1;
      for (uint32_t i = lane, j = 0; i < n_sys; i += 32, ++j) {
        if ((taken >> j) & 1u) continue;
        uint2 e = ld_key(i);
        uint32_t id = e.y & kIdMask;
        if (bi < 0 || (int)e.x < bk || ((int)e.x == bk && id < bid)) { bk = (int)e.x; bid = id; bi = (int)i; }
      }
      int mk = __reduce_min_sync(MIG_FULL, bi >= 0 ? bk : MIG_INF);
      uint32_t cm = __ballot_sync(MIG_FULL, bi >= 0 && bk == mk);
      if (cm & (cm - 1)) {
        uint32_t mid = __reduce_min_sync(MIG_FULL, (bi >= 0 && bk == mk) ? bid : 0xFFFFFFFFu);
        cm = __ballot_sync(MIG_FULL, bi >= 0 && bk == mk && bid == mid);
      }
      int wl = __ffs((int)cm) - 1;
      uint32_t b = (uint32_t)__shfl_sync(MIG_FULL, bi, wl);
      if (lane == wl) taken |= 1u << (b >> 5);
      uint4 E = ld_entry(b);                                   // broadcast: {skey, meta, rem, due}
      uint32_t cls = (E.y >> 20) & 15u;
      // --- slice choice by the 7 slice lanes
      bool mine = (avail >> lane) & 1u;
      int r = mine ? rd_magic((int)E.z, hot.speed[cls * 5 + max(sidx_of(sl_size), 0)]) : MIG_INF;
      uint32_t pick = 0;
      if (algo == MIG_ALGO_EDF_SS) {                           // slowest slice that still meets the deadline
        bool feas = mine && (r <= (int)E.w - t);
        int rmax = __reduce_max_sync(MIG_FULL, feas ? r : -1);
        if (rmax >= 0) pick = __ballot_sync(MIG_FULL, feas && r == rmax);
      }
      if (!pick) {                                             // fastest available slice
        int rmin = __reduce_min_sync(MIG_FULL, r);
        pick = __ballot_sync(MIG_FULL, mine && r == rmin);
      }
      int s;
      if (pick & (pick - 1)) {                                 // ties -> smaller size, then lower slot (reading #4)
        int k2 = __reduce_min_sync(MIG_FULL, ((pick >> lane) & 1u) ? sl_size * 8 + lane : MIG_INF);
        s = k2 & 7;
      } else s = __ffs((int)pick) - 1;
      avail &= ~(1u << s);
      if (lane == s) { new_pos = (int)b; new_rem = (int)E.z; new_due = (int)E.w; new_id = E.y & kIdMask; new_cls = cls; new_r = r; }
      if (lane == K) { asg_slot = s; asg_old1 = (int)((E.y >> 28) & 7u); asg_rem = (int)E.z; asg_id = E.y & kIdMask; asg_pos = b; asg_meta = E.y; }
      ++K;
    }
    // --- diff against the previous assignment: PREEMPT ascending old slot, START in priority order
    bool pre = busy && new_pos != sl_pos;
    uint32_t pm = __ballot_sync(MIG_FULL, pre);
    count(C_PREEMPT, __popc(pm));
    for (uint32_t m = pm; m; m &= m - 1) {
      int p = __ffs((int)m) - 1;
      emit(MIG_EV_PREEMPT, p, (uint32_t)size_at(p), __shfl_sync(MIG_FULL, rj_id, p), __shfl_sync(MIG_FULL, rj_rem, p));
    }
    bool st = lane < K && asg_slot + 1 != asg_old1;
    uint32_t sm = __ballot_sync(MIG_FULL, st);
    count(C_START, __popc(sm));
    for (uint32_t m = sm; m; m &= m - 1) {
      int r_ = __ffs((int)m) - 1;
      int s = __shfl_sync(MIG_FULL, asg_slot, r_);
      emit(MIG_EV_START, s, (uint32_t)size_at(s), __shfl_sync(MIG_FULL, asg_id, r_), __shfl_sync(MIG_FULL, asg_rem, r_));
    }
    // --- commit: slot field of the entries, then the slice lanes adopt their jobs
    if (pre) *entry_word((uint32_t)sl_pos, 1) &= ~(7u << 28);
    __syncwarp();
    if (st) *entry_word(asg_pos, 1) = (asg_meta & ~(7u << 28)) | ((uint32_t)(asg_slot + 1) << 28);
    __syncwarp();
    if (new_pos != sl_pos) {
      sl_pos = new_pos;
      if (new_pos >= 0) {
        rj_id = new_id; rj_rem = new_rem; rj_due = new_due;
        rj_v = hot.speed[new_cls * 5 + sidx_of(sl_size)].x;
        rj_ctime = t + new_r;
      }
    }
    update_power();
    compute_next_crit();
  }

  // remove entry `pos` (swap with the last); slice lanes tracking the last entry follow it
  __device__ __forceinline__ void remove_entry(uint32_t pos) {
    uint32_t last = n_sys - 1;
    if (pos != last) {
      uint4 e = ld_entry(last);
      __syncwarp();
      if (lane == 0) st_entry(pos, e);
      if (sl_pos == (int)last) sl_pos = (int)pos;
    }
    n_sys = last;
    __syncwarp();
  }

  // ------------------------------------------------------------------ event loop
  __device__ __forceinline__ void run_until(int t_end, bool drain) {
    for (;;) {
      if (drain && n_sys == 0) break;                         // energy stops at the last completion (reading #12)
      // 2. next event time
      int cand = MIG_INF;
      if (sl_pos >= 0) cand = rj_ctime;
      if (sl_size && sl_down) cand = min(cand, sl_upat);
      int tn = min(__reduce_min_sync(MIG_FULL, cand), t_end);
      if (look_valid) tn = min(tn, look_tick);
      tn = min(tn, next_crit);
      int dt = tn - t;
      e_ep += (long long)P * dt;
      busy_ep += (long long)U * dt;
      if (sl_pos >= 0 && dt) { rj_rem -= dt * (int)rj_v; *entry_word((uint32_t)sl_pos, 2) = (uint32_t)rj_rem; }
      t = tn;
      __syncwarp();
      // 3. same-tick order (reading #10): completions, slice-ups, arrivals, critical laxity, then ONE reschedule
      bool happened = false;
      uint32_t cm = __ballot_sync(MIG_FULL, sl_pos >= 0 && rj_rem <= 0);
      for (uint32_t m = cm; m; m &= m - 1) {                  // (i) completions, ascending slot
        int p = __ffs((int)m) - 1;
        int due = __shfl_sync(MIG_FULL, rj_due, p);
        uint32_t pos = (uint32_t)__shfl_sync(MIG_FULL, sl_pos, p);
        int tard = max(t - due, 0);                           // l_j = max(c_j - d_j, 0)
        emit(MIG_EV_COMPLETE, p, (uint32_t)size_at(p), __shfl_sync(MIG_FULL, rj_id, p), tard);
        tard_ep += tard;
        count(C_COMPLETED); count(C_TARDY, tard > 0 ? 1u : 0u);
        if (lane == p) sl_pos = -1;
        remove_entry(pos);
        happened = true;
      }
      uint32_t um = __ballot_sync(MIG_FULL, sl_size && sl_down && sl_upat == t);
      for (uint32_t m = um; m; m &= m - 1) {                  // (ii) slices coming up
        int p = __ffs((int)m) - 1;
        emit(MIG_EV_SLICE_UP, p, (uint32_t)size_at(p), 0xFFFFFFFFu, 0);
        if (lane == p) sl_down = 0;
        happened = true;
      }
      const uint32_t n_before = n_sys;
      while (look_valid && look_tick == t) {                  // (iii) arrivals, candidate order
        count(C_ARRIVED);
        if (n_sys == a.cap) {                                 // queue cap (BASELINE C3/C5)
          emit(MIG_EV_DROP, 0xFF, look_cls, look_id, look_due);
          count(C_DROPPED);
        } else {
          int sk = skey_of(look_due, look_work, look_cls);
          if (lane == 0) st_entry(n_sys, make_uint4((uint32_t)sk, look_id | (look_cls << 20), (uint32_t)look_work, (uint32_t)look_due));
          n_sys++;
          emit(MIG_EV_ARRIVE, 0xFF, look_cls, look_id, look_due);
          if (lane == 16 + C_SYSMAX) cnt_ep = max(cnt_ep, n_sys);
        }
        happened = true;
        gen_next();
      }
      __syncwarp();
      if (next_crit == t) {                                   // (iv) critical laxity, ascending id
        int last_id = -1;
        for (;;) {
          uint32_t bid = 0xFFFFFFFFu; int bi = -1;
          for (uint32_t i = lane; i < n_before; i += 32) {
            uint2 e = ld_key(i);
            uint32_t id = e.y & kIdMask;
            bool q = ((e.y >> 28) & 7u) == 0u && ((e.y >> 24) & 15u) < a.crit_max && (int)e.x - a.theta == t && (int)id > last_id;
            if (q && id < bid) { bid = id; bi = (int)i; }
          }
          uint32_t mid = __reduce_min_sync(MIG_FULL, bid);
          if (mid == 0xFFFFFFFFu) break;
          int wl = __ffs((int)__ballot_sync(MIG_FULL, bid == mid)) - 1;
          uint32_t b = (uint32_t)__shfl_sync(MIG_FULL, bi, wl);
          uint4 E = ld_entry(b);
          uint32_t cc = ((E.y >> 24) & 15u) + 1u;
          __syncwarp();
          if (lane == 0) *entry_word(b, 1) = (E.y & ~(15u << 24)) | (cc << 24);
          __syncwarp();
          emit(MIG_EV_CRIT, 0xFF, cc, mid, (int)E.w);
          count(C_CRIT);
          last_id = (int)mid;
          happened = true;
        }
      }
      if (happened) reschedule();                             // (v)
      if (t == t_end) break;
    }
  }

  // ------------------------------------------------------------------ repartition (readings #13, #14)
  __device__ __forceinline__ void prologue(uint32_t action) {
    repartitioned = 0;
    if (action >= a.n_configs) { status |= MIG_ST_BAD_ACTION; return; }
    if ((int)action == cfg) return;                           // "remain on the current configuration": no cost, no event
    uint32_t newsizes = hot.cfg_pack[action];
    int mynew = lane < kSlots ? (int)((newsizes >> (4 * lane)) & 15u) : 0;
    bool destroyed = sl_size && sl_size != mynew;
    uint32_t pm = __ballot_sync(MIG_FULL, destroyed && sl_pos >= 0);
    count(C_PREEMPT, __popc(pm));
    for (uint32_t m = pm; m; m &= m - 1) {                    // jobs on destroyed slices go back to waiting
      int p = __ffs((int)m) - 1;
      emit(MIG_EV_PREEMPT, p, (uint32_t)size_at(p), __shfl_sync(MIG_FULL, rj_id, p), __shfl_sync(MIG_FULL, rj_rem, p));
    }
    if (destroyed && sl_pos >= 0) { *entry_word((uint32_t)sl_pos, 1) &= ~(7u << 28); sl_pos = -1; }
    if (sl_size != mynew) {                                   // same (start, size) in both rows keeps job and up_at
      sl_size = mynew; sl_pos = -1; sl_down = 0; sl_upat = 0;
      if (mynew && a.downtime_s > 0) { sl_down = 1; sl_upat = t + a.downtime_s; }
    }
    int old = cfg;
    cfg = (int)action; cfg_sizes = newsizes;
    e_ep += a.repart_energy;
    repartitioned = 1; count(C_REPART);
    emit(MIG_EV_REPART, 0xFF, ((uint32_t)old << 8) | action, 0xFFFFFFFFu, 0);
    __syncwarp();
    if (algo >= MIG_ALGO_LLF) {                               // laxity keys are measured against the configuration
      for (uint32_t i = lane; i < n_sys; i += 32) {
        uint4 E = ld_entry(i);
        *entry_word(i, 0) = (uint32_t)skey_of((int)E.w, (int)E.z, (E.y >> 20) & 15u);
      }
      __syncwarp();
    }
    reschedule();
  }

  // ------------------------------------------------------------------ records
  __device__ __forceinline__ void begin_span() {
    e_ep = 0; tard_ep = 0; busy_ep = 0;
    cnt_ep = (lane == 16 + C_SYSMAX) ? n_sys : 0u;
    repartitioned = 0;
  }

  // fold the span into the totals; optionally store the 64-byte record (lanes 0..15, one 4-byte word each)
  __device__ __forceinline__ void close_record(mig_epoch_rec_t *r) {
    __syncwarp();
    if (lane >= 16 && lane < 26) {
      int c = lane - 16;
      uint32_t old = ws[WS_CNT + c];
      ws[WS_CNT + c] = (c == C_SYSMAX) ? max(old, cnt_ep) : old + cnt_ep;
    }
    if (lane == 0) {
      unsigned long long *tot = reinterpret_cast<unsigned long long *>(&ws[WS_TOT]);
      tot[0] += (unsigned long long)e_ep; tot[1] += (unsigned long long)tard_ep; tot[2] += (unsigned long long)busy_ep;
    }
    __syncwarp();
    if (!r) return;
    uint32_t c[10];
#pragma unroll
    for (int i = 0; i < 10; ++i) c[i] = __shfl_sync(MIG_FULL, cnt_ep, 16 + i);
    uint32_t n_run = __popc(__ballot_sync(MIG_FULL, sl_pos >= 0));
    uint32_t w = 0;
    switch (lane) {
      case 0: w = (uint32_t)e_ep; break;
      case 1: w = (uint32_t)((unsigned long long)e_ep >> 32); break;
      case 2: w = (uint32_t)tard_ep; break;
      case 3: w = (uint32_t)((unsigned long long)tard_ep >> 32); break;
      case 4: w = h_lo; break;
      case 5: w = h_hi; break;
      case 6: w = (uint32_t)busy_ep; break;
      case 7: w = (uint32_t)t; break;
      case 8: w = c[C_EVENTS]; break;
      case 9: w = (c[C_ARRIVED] & 0xFFFFu) | (c[C_COMPLETED] << 16); break;
      case 10: w = (c[C_DROPPED] & 0xFFFFu) | (c[C_TARDY] << 16); break;
      case 11: w = (c[C_PREEMPT] & 0xFFFFu) | (c[C_START] << 16); break;
      case 12: w = (c[C_CRIT] & 0xFFFFu) | (n_sys << 16); break;
      case 13: w = (uint32_t)cfg | ((uint32_t)repartitioned << 8) | ((status & 0xFFu) << 16) | (n_run << 24); break;
      case 14: w = c[C_SYSMAX]; break;
      default: w = 0; break;
    }
    if (lane < 16) reinterpret_cast<uint32_t *>(r)[lane] = w;
  }

  __device__ __forceinline__ void store_totals(mig_totals_t *o) {
    __syncwarp();
    uint32_t w = 0;
    if (lane < 8) w = (lane == 4) ? h_lo : (lane == 5) ? h_hi : ws[WS_TOT + (lane < 4 ? lane : lane - 2)];
    else if (lane < 18) w = ws[WS_CNT + (lane - 8)];
    else if (lane == 18) w = (uint32_t)t;
    else if (lane == 19) w = status;
    // word order of mig_totals_t: energy(0,1) tard(2,3) hash(4,5) busy(6,7) n_jobs..n_sys_max(8..17) t_end(18) status(19)
    if (lane < 20) reinterpret_cast<uint32_t *>(o)[lane] = w;
  }

  // ------------------------------------------------------------------ state vector
  __device__ __forceinline__ void observe(float *out) {
    __syncwarp();
    if (lane < 16) ws[WS_CLS + lane] = 0;
    __syncwarp();
    for (uint32_t i = lane; i < n_sys; i += 32) {
      uint32_t m = ld_key(i).y;
      if (((m >> 28) & 7u) == 0u) atomicAdd(&ws[WS_CLS + ((m >> 20) & 15u)], 1u);
    }
    __syncwarp();
    float lo = 0.f, hi = 0.f;                                  // x[lane], x[lane + 32]
    if (lane < 16) lo = (float)ws[WS_CLS + lane];
    float occ = sl_down ? 0.5f : (sl_pos >= 0 ? 1.0f : 0.0f);
#pragma unroll
    for (int p = 0; p < kSlots; ++p) {
      int g = __shfl_sync(MIG_FULL, sl_size, p);
      float v = __shfl_sync(MIG_FULL, occ, p);
      int q = lane - 16;
      if (g && q >= p && q < p + g && q < kSlots) lo = v;
      if (lane == 23 + p) lo = (float)g * 0.125f;
    }
    int hour = (t / 3600) % 24;
    if (lane == 30 + hour) lo = 1.0f;
    if (lane + 32 == 30 + hour) hi = 1.0f;
    uint32_t n_run = __popc(__ballot_sync(MIG_FULL, sl_pos >= 0));
    if (lane == 22) hi = (float)(n_sys - n_run) * (1.0f / 64.0f);
    if (lane == 23) hi = (float)n_run * 0.125f;
    uint32_t taken = 0;
    for (int m = 0; m < 3 && (uint32_t)m < n_sys; ++m) {        // first m = 3 jobs in (due, id) order
      int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu; int bi = -1;
      for (uint32_t i = lane, j = 0; i < n_sys; i += 32, ++j) {
        if ((taken >> j) & 1u) continue;
        uint4 E = ld_entry(i);
        uint32_t id = E.y & kIdMask;
        if (bi < 0 || (int)E.w < bk || ((int)E.w == bk && id < bid)) { bk = (int)E.w; bid = id; bi = (int)i; }
      }
      int mk = __reduce_min_sync(MIG_FULL, bi >= 0 ? bk : MIG_INF);
      uint32_t mid = __reduce_min_sync(MIG_FULL, (bi >= 0 && bk == mk) ? bid : 0xFFFFFFFFu);
      int wl = __ffs((int)__ballot_sync(MIG_FULL, bi >= 0 && bk == mk && bid == mid)) - 1;
      uint32_t b = (uint32_t)__shfl_sync(MIG_FULL, bi, wl);
      if (lane == wl) taken |= 1u << (b >> 5);
      uint4 E = ld_entry(b);
      int d = max(-32768, min(32767, (int)E.w - t));
      int mean = min(rd_cfg((int)E.z, (E.y >> 20) & 15u, true), 32767);
      if (lane == 24 + m) hi = (float)d * (1.0f / 4096.0f);
      if (lane == 27 + m) hi = (float)mean * (1.0f / 4096.0f);
    }
    if (lane == 30) hi = (float)ws[WS_DROPS] * (1.0f / 64.0f);
    if (lane == 31) hi = 1.0f;
    out[lane] = lo; out[lane + 32] = hi;
  }

  // ------------------------------------------------------------------ init / load / save
  __device__ __forceinline__ void set_config(int c) {
    cfg = c; cfg_sizes = hot.cfg_pack[c];
    sl_size = lane < kSlots ? size_at(lane) : 0;
    sl_down = 0; sl_upat = 0; sl_pos = -1;
  }

  __device__ __forceinline__ void init(uint32_t env_local) {
    algo = a.algo[env_local] & 3; t = 0; epoch = 0; status = 0; n_sys = 0;
    h_lo = 0x84222325u; h_hi = 0xcbf29ce4u;                   // FNV-1a-64 offset basis
    uint32_t c0 = a.cfg0[env_local];
    if (c0 >= a.n_configs) { c0 = 0; status |= MIG_ST_BAD_ACTION; }
    set_config((int)c0);
    rj_rem = 0; rj_due = 0; rj_ctime = 0; rj_id = 0; rj_v = 0;
    g_k = 0; g_T = 0; g_pending = 0; n_accepted = 0; g_done = 0; g_kbase = 0;
    g_tick = 0; g_work = 0; g_due = 0; g_cls = 0;
    next_crit = MIG_INF; n_trace = 0;
    __syncwarp();
    ws[lane] = 0; ws[lane + 32] = 0;
    __syncwarp();
    begin_span();
    update_power();
    gen_next();
  }

  __device__ __forceinline__ void save(uint32_t env_local) {
    __syncwarp();
    uint32_t lf = (uint32_t)look_valid;
    uint32_t w0 = 0, w1 = 0;
    switch (lane) {
      case 7: w0 = (uint32_t)t; break;
      case 8: w0 = (uint32_t)epoch | ((uint32_t)cfg << 8) | ((uint32_t)algo << 16) | (status << 24); break;
      case 9: w0 = n_sys; break;
      case 10: w0 = h_lo; break;
      case 11: w0 = h_hi; break;
      case 12: w0 = g_kbase; break;
      case 13: w0 = ws[WS_TBASE]; break;
      case 14: w0 = ws[WS_TBASE + 1]; break;
      case 15: w0 = g_pending; break;
      case 16: w0 = n_accepted; break;
      case 17: w0 = g_done; break;
      case 18: w0 = ws[WS_ISCRIPT]; break;
      case 19: w0 = ws[WS_DROPS]; break;
      case 20: case 21: case 22: case 23: case 24: case 25: w0 = ws[WS_TOT + lane - 20]; break;
      case 26: w0 = lf; break;
      case 27: w0 = (uint32_t)look_tick; break;
      case 28: w0 = look_cls; break;
      case 29: w0 = (uint32_t)look_work; break;
      case 30: w0 = (uint32_t)look_due; break;
      case 31: w0 = look_id; break;
      default: w0 = (uint32_t)sl_upat; break;                 // lanes 0..6
    }
    if (lane < kSlots) w1 = (uint32_t)sl_size | ((uint32_t)sl_down << 8) | ((uint32_t)(sl_pos + 1) << 16);
    else if (lane >= 16 && lane < 26) w1 = ws[WS_CNT + lane - 16];
    else if (lane == 7) w1 = (uint32_t)g_k;
    else if (lane == 8) w1 = (uint32_t)g_T;
    else if (lane == 9) w1 = (uint32_t)(g_T >> 32);
    uint32_t *h = a.hdr + (size_t)env_local * kHeaderWords;
    h[lane] = w0; h[lane + 32] = w1;
    uint32_t ns = min(n_sys, a.smem_entries);
    for (uint32_t i = lane; i < ns; i += 32) gtab[i] = stab[i];
  }

  __device__ __forceinline__ void load(uint32_t env_local) {
    const uint32_t *h = a.hdr + (size_t)env_local * kHeaderWords;
    uint32_t w0 = h[lane], w1 = h[lane + 32];
#define MIG_U(l) __shfl_sync(MIG_FULL, w0, l)
    t = (int)MIG_U(7);
    uint32_t pk = MIG_U(8);
    epoch = pk & 0xFF; cfg = (pk >> 8) & 0xFF; algo = (pk >> 16) & 0xFF; status = pk >> 24;
    n_sys = MIG_U(9); h_lo = MIG_U(10); h_hi = MIG_U(11);
    g_kbase = MIG_U(12);
    uint32_t tb_lo = MIG_U(13), tb_hi = MIG_U(14);
    uint32_t pend = MIG_U(15);
    n_accepted = MIG_U(16); g_done = MIG_U(17);
    uint32_t iscript = MIG_U(18), drops = MIG_U(19);
    look_valid = (int)MIG_U(26); look_tick = (int)MIG_U(27); look_cls = MIG_U(28); look_work = (int)MIG_U(29);
    look_due = (int)MIG_U(30); look_id = MIG_U(31);
#undef MIG_U
    g_k = __shfl_sync(MIG_FULL, w1, 7);
    g_T = (unsigned long long)__shfl_sync(MIG_FULL, w1, 8) | ((unsigned long long)__shfl_sync(MIG_FULL, w1, 9) << 32);
    cfg_sizes = hot.cfg_pack[cfg];
    sl_size = 0; sl_down = 0; sl_upat = 0; sl_pos = -1;
    if (lane < kSlots) { sl_upat = (int)w0; sl_size = w1 & 0xFF; sl_down = (w1 >> 8) & 0xFF; sl_pos = (int)(w1 >> 16) - 1; }
    __syncwarp();
    ws[lane] = 0; ws[lane + 32] = 0;
    __syncwarp();
    if (lane >= 16 && lane < 26) ws[WS_CNT + lane - 16] = w1;
    if (lane >= 20 && lane < 26) ws[WS_TOT + lane - 20] = w0;
    if (lane == 0) { ws[WS_TBASE] = tb_lo; ws[WS_TBASE + 1] = tb_hi; ws[WS_DROPS] = drops; ws[WS_ISCRIPT] = iscript; }
    uint32_t ns = min(n_sys, a.smem_entries);
    for (uint32_t i = lane; i < ns; i += 32) stab[i] = gtab[i];
    __syncwarp();
    g_tick = 0; g_work = 0; g_due = 0; g_cls = 0; g_pending = 0;
    if (pend) {                                              // rebuild the candidates of the batch in flight
      uint32_t gk = g_k; unsigned long long gT = g_T; uint32_t gd = g_done;
      gen_batch(g_kbase, (unsigned long long)tb_lo | ((unsigned long long)tb_hi << 32));
      g_k = gk; g_T = gT; g_done = gd; g_pending = pend;
    }
    rj_rem = 0; rj_due = 0; rj_ctime = 0; rj_id = 0; rj_v = 0;
    if (sl_pos >= 0) {                                       // running job: t + ceil(rem / v) never drifts
      uint4 E = ld_entry((uint32_t)sl_pos);
      uint4 sp = hot.speed[((E.y >> 20) & 15u) * 5 + sidx_of(sl_size)];
      rj_id = E.y & kIdMask; rj_rem = (int)E.z; rj_due = (int)E.w; rj_v = sp.x;
      rj_ctime = t + rd_magic(rj_rem, sp);
    }
    n_trace = 0;
    begin_span();
    update_power();
    compute_next_crit();
  }

  // ------------------------------------------------------------------ one decision epoch
  __device__ __forceinline__ void step(uint32_t env_local, uint32_t action) {
    const int k = epoch;
    begin_span();
    prologue(action);
    run_until((k + 1) * a.epoch_s, false);
    long long dE = e_ep, dT = tard_ep;
    uint32_t drops = __shfl_sync(MIG_FULL, cnt_ep, 16 + C_DROPPED);
    __syncwarp();
    if (lane == 0) ws[WS_DROPS] = drops;
    close_record(a.recs ? a.recs + (size_t)(k - a.rec_k0) * a.rec_stride + env_local : nullptr);
    if (k == a.n_epochs - 1) {                                // 4. drain (reading #11)
      begin_span();
      run_until(a.t_limit_s, true);
      if (n_sys > 0) status |= MIG_ST_TRUNCATED;
      dE += e_ep; dT += tard_ep;
      close_record(a.drain_rec ? a.drain_rec + env_local : nullptr);
    }
    epoch = k + 1;
    if (lane == 0) {
      if (a.energy_out) a.energy_out[env_local] = dE;
      if (a.tard_out) a.tard_out[env_local] = dT;
      if (a.reward_out)                                       // two fp32 products, one add, negate; no contraction
        a.reward_out[env_local] = -__fadd_rn(__fmul_rn(a.w_energy, __ll2float_rn(dE)), __fmul_rn(a.w_tardy, __ll2float_rn(dT)));
    }
  }
};

template <bool TRACE>
__global__ void __launch_bounds__(kWarpsPerCta * 32, 4) sim_kernel(const SimArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HotTables &hot = *reinterpret_cast<HotTables *>(smem_raw);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  {
    const DevTables *tb = a.tab;
    for (int i = threadIdx.x; i < MIG_MAX_CLASSES * 5; i += blockDim.x) hot.speed[i] = tb->speed[i];
    for (int i = threadIdx.x; i < MIG_MAX_CONFIGS; i += blockDim.x) hot.cfg_pack[i] = tb->cfg_pack[i];
    if (threadIdx.x < 8) { hot.curve[threadIdx.x] = tb->curve[threadIdx.x]; hot.p_idle[threadIdx.x] = tb->p_idle[threadIdx.x]; hot.p_busy[threadIdx.x] = tb->p_busy[threadIdx.x]; }
  }
  __syncthreads();
  const size_t per_warp = WS_WORDS * 4 + (size_t)a.smem_entries * 16;
  unsigned char *base = smem_raw + ((sizeof(HotTables) + 15) & ~(size_t)15) + (size_t)warp * per_warp;
  uint32_t *ws = reinterpret_cast<uint32_t *>(base);
  uint4 *stab = reinterpret_cast<uint4 *>(base + WS_WORDS * 4);
  Env<TRACE> e(a, hot, ws, stab, lane);
  for (;;) {
    uint32_t idx = 0;
    if (lane == 0) idx = atomicAdd(a.counter, 1u);
    idx = __shfl_sync(MIG_FULL, idx, 0);
    if (idx >= a.n_envs) break;
    const uint32_t env = a.env_first + idx;
    e.env_g = a.env_base + env;
    e.gtab = a.tab_override ? a.tab_override : a.jobtab + (size_t)env * a.cap;
    if (a.from_init) e.init(env); else e.load(env);
    for (int s = 0; s < a.n_steps && e.epoch < a.n_epochs; ++s) {
      uint32_t action = (uint32_t)e.cfg;                                            // STATIC: stay
      if (a.policy == MIG_POLICY_TABLE) {                                           // load bucket
        uint32_t b = e.n_sys == 0 ? 0u : (e.n_sys < 8 ? 1u : (e.n_sys < 64 ? 2u : 3u));
        action = a.table[((size_t)env * a.n_epochs + e.epoch) * 4 + b];
      } else if (a.actions) {
        action = a.actions[(size_t)idx * a.act_stride_env + (size_t)s * a.act_stride_k];
      }
      e.step(TRACE ? 0u : env, action);
    }
    if (a.state_out) e.observe(a.state_out + (size_t)(TRACE ? 0u : env) * MIG_STATE_DIM);
    if (a.totals) {                                           // totals so far (hash and t are live values)
      e.store_totals(a.totals + (TRACE ? 0u : env));
    }
    if (a.save) e.save(env);
    if (TRACE && a.trace_n && lane == 0) *a.trace_n = e.n_trace;
    __syncwarp();
  }
}

}  // namespace migsim
