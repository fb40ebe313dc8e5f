// sim_thread.cuh -- the rollout kernel with ONE THREAD PER ENVIRONMENT (mig_sim_set_tile(s, 1)).
//
// Why: the warp-tile kernel of sim_device.cuh spends most of its issue slots on cross-lane plumbing (butterfly
// reductions, ballots, broadcasts) for queues that hold about a dozen jobs and a GPU that has 7 slots.  With one
// environment per lane there is NO cross-lane traffic at all: every lane runs the serial event loop of DESIGN.md 3.3 on
// its own environment and a warp instruction advances 32 environments at once; the price is branch divergence between
// lanes, which the hardware reconverges (profiles/ has the measured threads-per-instruction).  It needs enough
// environments to fill the machine (one resident wave = 148 SMs x 448 threads = 66 304 environments), which is what
// the heavy batches (BASELINE C5: 65 536) have; small batches stay on the 8-lane tiles.
//
// Per-thread data lives in shared memory, interleaved by thread (word w of thread tid at base[w * NT + tid], so every
// access of a warp is bank-conflict-free whatever index each lane uses):
//   * slice table: table position and speed of the running job, up_at, per slot;
//   * job table {skey, meta | rem, due} (16 B / job), first `smem_entries` entries, overflow in global memory;
//   * the counters of the current record span and the reschedule's assignment scratch.
// Scalars (time, hash, energy, generator, look-ahead arrival) live in registers.  The results are bit-identical to the
// tile kernels and to the oracle (tests/test_gpu_parity.py); no code is shared with oracle/.
#pragma once
#include "sim_device.cuh"

namespace migsim {

constexpr int kThreadCta = 64;   // threads (= environments) per CTA of the thread-per-environment kernel

// per-thread 32-bit words ahead of the job table
enum { TW_POS = 0 /* 7: table index of the running job */, TW_V = 7 /* 7: its speed on the slice */, TW_UPAT = 14 /* 7 */,
       TW_CNT = 21 /* C_COUNT = 10 */, TW_SCR = 31 /* 16: assignment scratch / class counters */, TW_FIXED = 48 };
enum { SCR_ASG = 0 /* 7 */, SCR_R = 8 /* 7 */ };

// saved per-env header of this kernel (kHeaderWords words); the running totals H1_TOT / H1_CNT live here all the time
enum { H1_UPAT = 0 /* 7 */, H1_T = 7, H1_PK, H1_NSYS, H1_HLO, H1_HHI, H1_GK, H1_GT_LO, H1_GT_HI, H1_GDONE, H1_NACC, H1_ISCRIPT,
       H1_DROPS, H1_MASKS /* busy | down << 8 | fsz << 16 */, H1_TOT = 20 /* 6 */, H1_LOOKV = 26, H1_LOOKTICK, H1_LOOKCLS, H1_LOOKWORK,
       H1_LOOKDUE, H1_LOOKID, H1_POS = 32 /* 7 */, H1_CNT = 48 /* 10 */ };

struct HotTablesT {              // per CTA, shared memory
  HotTables h;
  uint32_t cfg_rank[MIG_MAX_CONFIGS];     // nibble p: rank of the slice starting at slot p in (size, slot) order (reading #4)
  uint32_t cfg_slot_of[MIG_MAX_CONFIGS];  // nibble r: start slot of the slice of rank r
  int32_t cfg_pidle[MIG_MAX_CONFIGS];     // sum of p_idle over the slices of the configuration
  uint32_t logT[257];
};

__host__ __device__ constexpr size_t thread_smem_bytes(uint32_t smem_entries, int nt) {
  return ((sizeof(HotTablesT) + 127) & ~(size_t)127) + (size_t)nt * (TW_FIXED + 4 * (size_t)smem_entries) * 4;
}

template <int NT, bool TRACE>
struct EnvT {
  // ------------------------------------------------------------------ environment state
  const SimArgs &a;
  const HotTablesT &hot;
  uint32_t *const fx;      // fixed words: fx[w * NT]
  uint2 *const tb;         // job table: {skey, meta} at tb[(2 * i) * NT], {rem, due} at tb[(2 * i + 1) * NT]
  uint4 *gtab;             // overflow part (and save area) in global memory, same entry index
  uint32_t *hdr;           // this env's saved header (running totals are kept there)
  const uint32_t S;        // entries held in shared memory
  uint32_t env_g;
  int t, t_end, epoch, cfg, algo; uint32_t status, n_sys, cfg_sizes, cfg_rank, slice_mask;
  uint32_t h_lo, h_hi;
  long long e_ep, tard_ep, busy_ep;
  int P, U, next_crit, next_done, next_up, repartitioned;
  uint32_t busy_mask, down_mask;
  uint32_t fsz;            // entries [0, fsz) of the job table are sorted by (key, id) and precede every other entry
  uint32_t g_k, g_done, n_accepted; unsigned long long g_T;
  int look_valid, look_tick, look_work, look_due; uint32_t look_cls, look_id;
  uint32_t n_trace, i_script, n_events;

  __device__ __forceinline__ EnvT(const SimArgs &a_, const HotTablesT &h_, uint32_t *fx_, uint2 *tb_)
      : a(a_), hot(h_), fx(fx_), tb(tb_), S(a_.smem_entries) {}

  // ------------------------------------------------------------------ job table access
  __device__ __forceinline__ uint2 ld_km(uint32_t i) const {
    return i < S ? tb[(2 * i) * NT] : *reinterpret_cast<const uint2 *>(&gtab[i]);
  }
  __device__ __forceinline__ uint2 ld_rd(uint32_t i) const {
    return i < S ? tb[(2 * i + 1) * NT] : *(reinterpret_cast<const uint2 *>(&gtab[i]) + 1);
  }
  __device__ __forceinline__ void st_entry(uint32_t i, uint2 km, uint2 rd) {
    if (i < S) { tb[(2 * i) * NT] = km; tb[(2 * i + 1) * NT] = rd; } else gtab[i] = make_uint4(km.x, km.y, rd.x, rd.y);
  }
  // word w of entry i: 0 skey, 1 meta, 2 rem, 3 due
  __device__ __forceinline__ uint32_t *entry_word(uint32_t i, int w) {
    if (i < S) return reinterpret_cast<uint32_t *>(&tb[(2 * i + (w >> 1)) * NT]) + (w & 1);
    return reinterpret_cast<uint32_t *>(&gtab[i]) + w;
  }
  __device__ __forceinline__ uint32_t &F(int w) { return fx[w * NT]; }
  __device__ __forceinline__ void count(int c, uint32_t n) { fx[(TW_CNT + c) * NT] += n; }

  // ------------------------------------------------------------------ sorted front of the job table
  // The reschedule needs the K <= 7 first jobs in (key, id) order.  Instead of K scans over the whole table, entries
  // [0, fsz), fsz <= kFront, are kept sorted and not larger than any other entry; the rest is unordered.  Arrivals are
  // sifted in, completions shift the front up, and a single pass over the rest refills the front when it runs short
  // (EDF keys never change; LLF / LALF keys of running jobs do, so those algorithms rebuild the front every time).
  static constexpr uint32_t kFront = 8;
  static __device__ __forceinline__ bool before(uint2 x, uint2 y) {          // (key, id) order; ties -> lower id (reading #5)
    return (int)x.x < (int)y.x || (x.x == y.x && (x.y & kIdMask) < (y.y & kIdMask));
  }
  // store an entry at `dst`; the slice running it follows
  __device__ __forceinline__ void put(uint32_t dst, uint2 km, uint2 rd) {
    st_entry(dst, km, rd);
    const uint32_t sl = (km.y >> 28) & 7u;
    if (sl) F(TW_POS + sl - 1) = dst;
  }
  // entries [0, len) are sorted and position len is free: place the entry so that [0, len] is sorted
  __device__ __forceinline__ void sift(uint32_t len, uint2 km, uint2 rd) {
    uint32_t j = len;
    while (j > 0) {
      const uint2 q = ld_km(j - 1);
      if (!before(km, q)) break;
      put(j, q, ld_rd(j - 1));
      --j;
    }
    put(j, km, rd);
  }
  __device__ __forceinline__ void insert_entry(uint2 km, uint2 rd) {
    const bool in_front = (fsz == n_sys && fsz < kFront) || (fsz > 0 && before(km, ld_km(fsz - 1)));
    if (!in_front) put(n_sys, km, rd);
    else if (fsz == kFront) { put(n_sys, ld_km(kFront - 1), ld_rd(kFront - 1)); sift(kFront - 1, km, rd); }
    else { if (fsz < n_sys) put(n_sys, ld_km(fsz), ld_rd(fsz)); sift(fsz, km, rd); fsz++; }
    n_sys++;
  }
  // make [0, min(kFront, n_sys)) the smallest entries, sorted: grow the front over what follows it, then one pass over the rest
  __device__ __forceinline__ void refill_front() {
    const uint32_t tgt = min(kFront, n_sys);
    while (fsz < tgt) { sift(fsz, ld_km(fsz), ld_rd(fsz)); fsz++; }
    if (n_sys <= kFront) return;
    uint2 worst = ld_km(kFront - 1);
    for (uint32_t i = kFront; i < n_sys; ++i) {
      const uint2 km = ld_km(i);
      if (before(km, worst)) {
        const uint2 rd = ld_rd(i);
        put(i, worst, ld_rd(kFront - 1));
        sift(kFront - 1, km, rd);
        worst = ld_km(kFront - 1);
      }
    }
  }

  // ------------------------------------------------------------------ trace
  __device__ __forceinline__ void fnv(uint32_t w) {
    // h = (h ^ w) * 0x100000001b3 (64-bit) in 32-bit pieces: h * (2^40 + 0x1b3)
    const uint32_t lo = h_lo ^ w;
    const unsigned long long p = (unsigned long long)lo * 0x1b3u;
    h_hi = (uint32_t)(p >> 32) + h_hi * 0x1b3u + (lo << 8);
    h_lo = (uint32_t)p;
  }
  __device__ __forceinline__ void emit(int type, int slot, uint32_t aux, uint32_t job, int value) {
    const uint32_t w1 = (uint32_t)type | ((uint32_t)(slot & 0xFF) << 8) | ((aux & 0xFFFFu) << 16);
    fnv((uint32_t)t); fnv(w1); fnv(job); fnv((uint32_t)value);
    if (TRACE) {
      if (a.trace && n_trace < a.trace_cap) reinterpret_cast<uint4 *>(a.trace)[n_trace] = make_uint4((uint32_t)t, w1, job, (uint32_t)value);
      n_trace++;
    }
    n_events++;
  }

  // ------------------------------------------------------------------ model
  __device__ __forceinline__ int size_at(int p) const { return (cfg_sizes >> (4 * p)) & 15; }
  __device__ __forceinline__ const uint4 &speed_of(uint32_t cls, int size) const { return hot.h.speed[cls * 5 + sidx_of(size)]; }

  // remaining duration against the configuration: fastest slice (LLF) or floor of the mean over all
  // slices of cfg, up or down (LALF; also the state vector's "average duration", L210)
  __device__ __forceinline__ int rd_cfg(int rem, uint32_t cls, bool mean) const {
    int best = MIG_INF, sum = 0, n = 0;
    for (uint32_t m = slice_mask; m; m &= m - 1) {
      const int r = rd_magic(rem, speed_of(cls, size_at(__ffs((int)m) - 1)));
      best = min(best, r); sum += r; ++n;
    }
    return mean ? sum / n : best;
  }
  __device__ __forceinline__ int skey_of(int due, int rem, uint32_t cls) const {
    if (algo < MIG_ALGO_LLF) return due;                                  // EDF: deadline
    return due - rd_cfg(rem, cls, algo == MIG_ALGO_LALF);                 // laxity + t (t is common to all jobs)
  }

  __device__ __forceinline__ void set_cfg_tables(int c) {
    cfg = c; cfg_sizes = hot.h.cfg_pack[c]; cfg_rank = hot.cfg_rank[c];
    uint32_t m = 0;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) m |= ((cfg_sizes >> (4 * p)) & 15u) ? (1u << p) : 0u;
    slice_mask = m;
  }

  // power and busy units from the slice table (a down slice counts idle)
  __device__ __forceinline__ void update_power() {
    int u = 0, pd = 0;
    for (uint32_t m = busy_mask; m; m &= m - 1) {
      const int g = size_at(__ffs((int)m) - 1);
      u += g; pd += hot.h.p_busy[g] - hot.h.p_idle[g];
    }
    U = u; P = hot.cfg_pidle[cfg] + pd + hot.h.curve[u & 7];
  }

  // ------------------------------------------------------------------ arrival generator (R2-R5)
  __device__ __forceinline__ uint32_t neglog2_q24(uint32_t w) const {
    const uint32_t m = w | 1u;
    const int lz = __clz((int)m);
    const uint32_t y = m << lz;
    const uint32_t i = (y >> 23) & 0xFFu, f = (y >> 7) & 0xFFFFu;
    const uint32_t T0 = hot.logT[i], T1 = hot.logT[i + 1];
    const uint32_t L = T0 + (uint32_t)(((unsigned long long)(T1 - T0) * f) >> 16);
    return ((uint32_t)(1 + lz) << 24) - L;
  }

  // advance the look-ahead to the next accepted arrival (or none): sequential thinning, one candidate per trip
  __device__ __forceinline__ void gen_next() {
    look_valid = 0;
    if (a.script) {                                                           // scripted arrivals (tests), kernel-uniform branch
      if (i_script < a.n_script) {
        const mig_job_t s = a.script[i_script];
        look_valid = 1; look_tick = s.arr; look_cls = s.cls; look_due = s.due;
        look_work = (int)((uint32_t)s.dur7 * hot.h.speed[s.cls * 5 + 4].x);
        look_id = i_script; n_accepted++; i_script++;
      }
      return;
    }
    const uint32_t limit = a.job_limit ? min(a.job_limit, MIG_MAX_JOBS) : MIG_MAX_JOBS;
    if (n_accepted >= limit) return;
    const DevTables *tb_ = a.tab;
    while (!g_done) {
      const uint32_t k = g_k++;
      const uint4 w = philox4x32_10(k, 0u, env_g, a.episode, a.k0, a.k1);    // stream 0: gap, accept, class, slack
      g_T += ((unsigned long long)neglog2_q24(w.x) * a.gap_scale) >> 24;
      const unsigned long long tick = g_T >> 16;
      if (tick >= (unsigned long long)a.day_s) { g_done = 1; break; }         // arrivals stop at the end of the day
      if (w.y > __ldg(&tb_->thr[(uint32_t)tick / 60u])) continue;              // Lewis-Shedler thinning
      uint32_t c = 0;
      for (uint32_t i = 0; i + 1 < a.n_classes; ++i) c += (w.z > __ldg(&tb_->class_cum[i])) ? 1u : 0u;
      const uint4 wd = philox4x32_10(k, 1u, env_g, a.episode, a.k0, a.k1);   // stream 1: duration
      const uint32_t qi = wd.x >> 26, f = (wd.x >> 16) & 0x3FFu;
      const int q0 = __ldg(&tb_->dur7_q[c * 65 + qi]), q1 = __ldg(&tb_->dur7_q[c * 65 + qi + 1]);
      const int dur7 = q0 + (int)(((long long)(q1 - q0) * (long long)f) >> 10);
      const uint32_t slack = __ldg(&tb_->slack_lo[c]) + __umulhi(w.w, __ldg(&tb_->slack_span[c]));
      unsigned long long rel = ((unsigned long long)(uint32_t)dur7 * slack) >> 10;
      if (rel < 1) rel = 1;
      look_tick = (int)tick; look_cls = c;
      look_work = (int)((uint32_t)dur7 * hot.h.speed[c * 5 + 4].x);
      look_due = (int)((long long)tick + (long long)rel);
      look_id = n_accepted++;
      look_valid = 1;
      break;
    }
  }

  // ------------------------------------------------------------------ reschedule
  // critical-laxity events (LLF / LALF): earliest t_crit = skey - theta > t over waiting jobs
  __device__ __forceinline__ void compute_next_crit() {
    int best = MIG_INF;
    if (algo >= MIG_ALGO_LLF)
      for (uint32_t i = 0; i < n_sys; ++i) {
        const uint2 e = ld_km(i);
        const int tc = (int)e.x - a.theta;
        const bool waiting = ((e.y >> 28) & 7u) == 0u;
        if (waiting && ((e.y >> 24) & 15u) < a.crit_max && tc > t) best = min(best, tc);
      }
    next_crit = best;
  }

  // every job in the system is re-evaluated: the K = min(up slices, jobs) first jobs in (key, id) order pick a slice each
  __device__ __forceinline__ void reschedule() {
    if (algo >= MIG_ALGO_LLF)                       // the keys of running jobs move with their remaining work
      for (uint32_t m = busy_mask; m; m &= m - 1) {
        const uint32_t pos = F(TW_POS + __ffs((int)m) - 1);
        const uint2 km = ld_km(pos), rdv = ld_rd(pos);
        *entry_word(pos, 0) = (uint32_t)skey_of((int)rdv.y, (int)rdv.x, (km.y >> 20) & 15u);
      }
    const uint32_t up = slice_mask & ~down_mask;    // every UP slice, occupied or not
    uint32_t avail = up;
    const int K = (int)min((uint32_t)__popc(up), n_sys);
    if (algo >= MIG_ALGO_LLF) fsz = 0;
    if (fsz < (uint32_t)K) refill_front();
    uint32_t keep = 0;
    for (int k = 0; k < K; ++k) {                   // entry k is the k-th job in (key, id) order
      const uint32_t bmeta = ld_km((uint32_t)k).y;
      const uint2 rdv = ld_rd((uint32_t)k);
      const int rem = (int)rdv.x, slack = (int)rdv.y - t;
      const uint32_t cls = (bmeta >> 20) & 15u;
      // --- slice choice: one composite key per rule, (r, rank) is unique per slice
      int fsb = MIG_INF, ssb = -1;
      for (uint32_t m = avail; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const int r = rd_magic(rem, speed_of(cls, size_at(p)));
        const int rk = (int)((cfg_rank >> (4 * p)) & 7u);
        fsb = min(fsb, (r << 3) | rk);                                    // fastest; ties -> smaller size, lower slot (reading #4)
        if (r <= slack) ssb = max(ssb, (r << 3) | (7 - rk));              // slowest that meets the deadline; same ties
      }
      const bool use_ss = algo == MIG_ALGO_EDF_SS && ssb >= 0;
      const int pick = use_ss ? ssb : fsb;
      const int rk = use_ss ? 7 - (pick & 7) : (pick & 7);
      const int s = (int)((hot.cfg_slot_of[cfg] >> (4 * rk)) & 7u);
      avail &= ~(1u << s);
      const bool moved = ((bmeta >> 28) & 7u) != (uint32_t)(s + 1);
      if (!moved) keep |= 1u << s;
      F(TW_SCR + SCR_ASG + k) = (uint32_t)s | (moved ? 0x8000u : 0u);
      F(TW_SCR + SCR_R + k) = (uint32_t)(pick >> 3);
    }
    // --- diff against the previous assignment: PREEMPT ascending old slot, START in priority order
    const uint32_t pm = busy_mask & ~keep;
    if (pm) {
      count(C_PREEMPT, __popc(pm));
      for (uint32_t m = pm; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const uint32_t pos = F(TW_POS + p);
        const uint2 km = ld_km(pos), rdv = ld_rd(pos);
        emit(MIG_EV_PREEMPT, p, (uint32_t)size_at(p), km.y & kIdMask, (int)rdv.x);
        *entry_word(pos, 1) = km.y & ~(7u << 28);
      }
    }
    uint32_t nb = 0; int nd = MIG_INF, u = 0, pd = 0, n_start = 0;
    for (int k = 0; k < K; ++k) {
      const uint32_t w = F(TW_SCR + SCR_ASG + k);
      const int r = (int)F(TW_SCR + SCR_R + k);
      const int s = (int)(w & 7u);
      const int g = size_at(s);
      nb |= 1u << s; nd = min(nd, t + r); u += g; pd += hot.h.p_busy[g] - hot.h.p_idle[g];
      if (w & 0x8000u) {
        const uint32_t pos = (uint32_t)k;
        const uint2 km = ld_km(pos), rdv = ld_rd(pos);
        emit(MIG_EV_START, s, (uint32_t)g, km.y & kIdMask, (int)rdv.x);
        *entry_word(pos, 1) = (km.y & ~(7u << 28)) | ((uint32_t)(s + 1) << 28);
        F(TW_POS + s) = pos;
        F(TW_V + s) = speed_of((km.y >> 20) & 15u, g).x;
        ++n_start;
      }
    }
    if (n_start) count(C_START, (uint32_t)n_start);
    busy_mask = nb; next_done = nd;
    U = u; P = hot.cfg_pidle[cfg] + pd + hot.h.curve[u & 7];
    compute_next_crit();
  }

  // remove entry `pos`: the sorted front closes up, the hole is filled with the last entry
  __device__ __forceinline__ void remove_entry(uint32_t pos) {
    uint32_t hole = pos;
    if (pos < fsz) {
      for (uint32_t j = pos; j + 1 < fsz; ++j) put(j, ld_km(j + 1), ld_rd(j + 1));
      hole = --fsz;
    }
    const uint32_t last = n_sys - 1;
    if (hole != last) put(hole, ld_km(last), ld_rd(last));
    n_sys = last;
  }

  // ------------------------------------------------------------------ event loop
  // one event time: advance to it, then the same-tick order of reading #10 and ONE reschedule
  __device__ __forceinline__ void event() {
    // 2. next event time (completions and slice-ups are kept as running minima)
    int tn = min(min(next_done, next_up), min(t_end, next_crit));
    if (look_valid) tn = min(tn, look_tick);
    const int dt = tn - t;
    e_ep += (long long)P * dt;
    busy_ep += (long long)U * dt;
    t = tn;
    uint32_t done = 0;
    if (dt)
      for (uint32_t m = busy_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        uint32_t *rp = entry_word(F(TW_POS + p), 2);
        const int rem = (int)*rp - dt * (int)F(TW_V + p);
        *rp = (uint32_t)rem;
        if (rem <= 0) done |= 1u << p;
      }
    bool happened = false;
    for (; done; done &= done - 1) {                                  // (i) completions, ascending slot
      const int p = __ffs((int)done) - 1;
      const uint32_t pos = F(TW_POS + p);
      const uint32_t id = ld_km(pos).y & kIdMask;
      const int tard = max(t - (int)ld_rd(pos).y, 0);                 // l_j = max(c_j - d_j, 0)
      emit(MIG_EV_COMPLETE, p, (uint32_t)size_at(p), id, tard);
      tard_ep += tard;
      count(C_COMPLETED, 1u);
      if (tard > 0) count(C_TARDY, 1u);
      busy_mask &= ~(1u << p);
      remove_entry(pos);
      happened = true;
    }
    if (next_up == t) {                                               // (ii) slices coming up, ascending slot
      int nu = MIG_INF;
      for (uint32_t m = down_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const int up = (int)F(TW_UPAT + p);
        if (up == t) { emit(MIG_EV_SLICE_UP, p, (uint32_t)size_at(p), MIG_NOJOB, 0); down_mask &= ~(1u << p); happened = true; }
        else nu = min(nu, up);
      }
      next_up = nu;
    }
    const uint32_t first_new = look_valid ? look_id : 0xFFFFFFFFu;   // ids are sequential: this tick's arrivals have id >= first_new
    while (look_valid && look_tick == t) {                            // (iii) arrivals, candidate order
      const bool drop = n_sys == a.cap;                               // queue cap (BASELINE C3/C5)
      count(C_ARRIVED, 1u);
      if (drop) count(C_DROPPED, 1u);
      else {
        insert_entry(make_uint2((uint32_t)skey_of(look_due, look_work, look_cls), look_id | (look_cls << 20)),
                     make_uint2((uint32_t)look_work, (uint32_t)look_due));
        if (n_sys > F(TW_CNT + C_SYSMAX)) F(TW_CNT + C_SYSMAX) = n_sys;
      }
      emit(drop ? MIG_EV_DROP : MIG_EV_ARRIVE, 0xFF, look_cls, look_id, look_due);
      happened = true;
      gen_next();
    }
    if (next_crit == t) {                                             // (iv) critical laxity, ascending id
      int last_id = -1;
      for (;;) {
        uint32_t bid = 0xFFFFFFFFu, bi = 0, bmeta = 0;
        for (uint32_t i = 0; i < n_sys; ++i) {                        // jobs present before this tick's arrivals (reading #23)
          const uint2 e = ld_km(i);
          const uint32_t id = e.y & kIdMask;
          const bool q = id < first_new && ((e.y >> 28) & 7u) == 0u && ((e.y >> 24) & 15u) < a.crit_max && (int)e.x - a.theta == t && (int)id > last_id;
          if (q && id < bid) { bid = id; bi = i; bmeta = e.y; }
        }
        if (bid == 0xFFFFFFFFu) break;
        const uint32_t cc = ((bmeta >> 24) & 15u) + 1u;
        *entry_word(bi, 1) = (bmeta & ~(15u << 24)) | (cc << 24);
        emit(MIG_EV_CRIT, 0xFF, cc, bid, (int)ld_rd(bi).y);
        count(C_CRIT, 1u);
        last_id = (int)bid;
        happened = true;
      }
    }
    if (happened) reschedule();                                       // (v)
  }

  // ------------------------------------------------------------------ repartition (readings #13, #14)
  __device__ __forceinline__ void prologue(uint32_t action) {
    repartitioned = 0;
    if (action >= a.n_configs) { status |= MIG_ST_BAD_ACTION; return; }
    if ((int)action == cfg) return;                           // "remain on the current configuration": no cost, no event
    const uint32_t newsizes = hot.h.cfg_pack[action];
    uint32_t changed = 0;                                     // slots whose (start, size) differs between the two rows
#pragma unroll
    for (int p = 0; p < kSlots; ++p) changed |= (((cfg_sizes ^ newsizes) >> (4 * p)) & 15u) ? (1u << p) : 0u;
    const uint32_t pm = busy_mask & changed;                  // jobs on destroyed slices go back to waiting
    if (pm) {
      count(C_PREEMPT, __popc(pm));
      for (uint32_t m = pm; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const uint32_t pos = F(TW_POS + p);
        const uint2 km = ld_km(pos);
        emit(MIG_EV_PREEMPT, p, (uint32_t)size_at(p), km.y & kIdMask, (int)ld_rd(pos).x);
        *entry_word(pos, 1) = km.y & ~(7u << 28);
      }
      busy_mask &= ~pm;
    }
    const int old = cfg;
    set_cfg_tables((int)action);
    down_mask &= ~changed;                                    // same (start, size) in both rows keeps job and up_at
    if (a.downtime_s > 0)
      for (uint32_t m = changed & slice_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        F(TW_UPAT + p) = (uint32_t)(t + a.downtime_s);
        down_mask |= 1u << p;
      }
    int nu = MIG_INF;
    for (uint32_t m = down_mask; m; m &= m - 1) nu = min(nu, (int)F(TW_UPAT + __ffs((int)m) - 1));
    next_up = nu;
    e_ep += a.repart_energy; repartitioned = 1;
    count(C_REPART, 1u);
    emit(MIG_EV_REPART, 0xFF, ((uint32_t)old << 8) | action, MIG_NOJOB, 0);
    if (algo >= MIG_ALGO_LLF)                                 // laxity keys are measured against the configuration
      for (uint32_t i = 0; i < n_sys; ++i) {
        const uint2 km = ld_km(i), rdv = ld_rd(i);
        *entry_word(i, 0) = (uint32_t)skey_of((int)rdv.y, (int)rdv.x, (km.y >> 20) & 15u);
      }
    reschedule();
  }

  // ------------------------------------------------------------------ records
  __device__ __forceinline__ void begin_span() {
    e_ep = 0; tard_ep = 0; busy_ep = 0; n_events = 0;
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) F(TW_CNT + i) = (i == C_SYSMAX) ? n_sys : 0u;
    repartitioned = 0;
  }

  // fold the span into the running totals (kept in the env's header); optionally store the 64-byte record
  __device__ __forceinline__ void close_record(mig_epoch_rec_t *r) {
    uint32_t c[C_COUNT];
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) c[i] = F(TW_CNT + i);
    c[C_EVENTS] = n_events;
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) hdr[H1_CNT + i] = (i == C_SYSMAX) ? max(hdr[H1_CNT + i], c[i]) : hdr[H1_CNT + i] + c[i];
    unsigned long long *tot = reinterpret_cast<unsigned long long *>(&hdr[H1_TOT]);
    tot[0] += (unsigned long long)e_ep; tot[1] += (unsigned long long)tard_ep; tot[2] += (unsigned long long)busy_ep;
    if (!r) return;
    uint4 *o = reinterpret_cast<uint4 *>(r);
    o[0] = make_uint4((uint32_t)e_ep, (uint32_t)((unsigned long long)e_ep >> 32), (uint32_t)tard_ep, (uint32_t)((unsigned long long)tard_ep >> 32));
    o[1] = make_uint4(h_lo, h_hi, (uint32_t)busy_ep, (uint32_t)t);
    o[2] = make_uint4(c[C_EVENTS], (c[C_ARRIVED] & 0xFFFFu) | (c[C_COMPLETED] << 16), (c[C_DROPPED] & 0xFFFFu) | (c[C_TARDY] << 16),
                      (c[C_PREEMPT] & 0xFFFFu) | (c[C_START] << 16));
    o[3] = make_uint4((c[C_CRIT] & 0xFFFFu) | (n_sys << 16),
                      (uint32_t)cfg | ((uint32_t)repartitioned << 8) | ((status & 0xFFu) << 16) | ((uint32_t)__popc(busy_mask) << 24),
                      c[C_SYSMAX], 0u);
  }

  // word order of mig_totals_t: energy(0,1) tard(2,3) hash(4,5) busy(6,7) n_jobs..n_sys_max(8..17) t_end(18) status(19)
  __device__ __forceinline__ void store_totals(mig_totals_t *o_) {
    uint4 *o = reinterpret_cast<uint4 *>(o_);
    o[0] = make_uint4(hdr[H1_TOT], hdr[H1_TOT + 1], hdr[H1_TOT + 2], hdr[H1_TOT + 3]);
    o[1] = make_uint4(h_lo, h_hi, hdr[H1_TOT + 4], hdr[H1_TOT + 5]);
    o[2] = make_uint4(hdr[H1_CNT], hdr[H1_CNT + 1], hdr[H1_CNT + 2], hdr[H1_CNT + 3]);
    o[3] = make_uint4(hdr[H1_CNT + 4], hdr[H1_CNT + 5], hdr[H1_CNT + 6], hdr[H1_CNT + 7]);
    o[4] = make_uint4(hdr[H1_CNT + 8], hdr[H1_CNT + 9], (uint32_t)t, status);
  }

  // ------------------------------------------------------------------ state vector
  __device__ __forceinline__ void observe(float *out) {
    float4 *o4 = reinterpret_cast<float4 *>(out);
#pragma unroll
    for (int w = 0; w < 16; ++w) F(TW_SCR + w) = 0u;
    for (uint32_t i = 0; i < n_sys; ++i) {                     // waiting jobs per class
      const uint32_t m = ld_km(i).y;
      if (((m >> 28) & 7u) == 0u) F(TW_SCR + (int)((m >> 20) & 15u)) += 1u;
    }
#pragma unroll
    for (int w = 0; w < 4; ++w)
      o4[w] = make_float4((float)F(TW_SCR + 4 * w), (float)F(TW_SCR + 4 * w + 1), (float)F(TW_SCR + 4 * w + 2), (float)F(TW_SCR + 4 * w + 3));
#pragma unroll
    for (int w = 4; w < 16; ++w) o4[w] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    const int n_run = __popc(busy_mask);
    for (uint32_t m = slice_mask; m; m &= m - 1) {
      const int p = __ffs((int)m) - 1, g = size_at(p);
      const float occ = ((down_mask >> p) & 1u) ? 0.5f : (((busy_mask >> p) & 1u) ? 1.0f : 0.0f);
      for (int q = 0; q < g; ++q) out[16 + p + q] = occ;        // slots covered by this slice
      out[23 + p] = (float)g * 0.125f;
    }
    out[30 + (t / 3600) % 24] = 1.0f;
    out[54] = (float)(n_sys - (uint32_t)n_run) * (1.0f / 64.0f);
    out[55] = (float)n_run * 0.125f;
    out[62] = (float)hdr[H1_DROPS] * (1.0f / 64.0f);
    out[63] = 1.0f;
    int pk = (int)0x80000000; uint32_t pid = 0;
    for (int m = 0; m < 3 && (uint32_t)m < n_sys; ++m) {        // first m = 3 jobs in (due, id) order
      int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu, bi = 0;
      for (uint32_t i = 0; i < n_sys; ++i) {
        const int due = (int)ld_rd(i).y; const uint32_t id = ld_km(i).y & kIdMask;
        const bool beyond = due > pk || (due == pk && id > pid);
        const bool better = due < bk || (due == bk && id < bid);
        if (beyond && better) { bk = due; bid = id; bi = i; }
      }
      const uint2 km = ld_km(bi), rdv = ld_rd(bi);
      const int d = max(-32768, min(32767, (int)rdv.y - t));
      const int mean = min(rd_cfg((int)rdv.x, (km.y >> 20) & 15u, true), 32767);
      out[56 + m] = (float)d * (1.0f / 4096.0f);
      out[59 + m] = (float)mean * (1.0f / 4096.0f);
      pk = bk; pid = bid;
    }
  }

  // ------------------------------------------------------------------ init / load / save
  __device__ __forceinline__ void init(uint32_t env_local) {
    algo = a.algo[env_local] & 3; t = 0; epoch = 0; status = 0; n_sys = 0;
    h_lo = 0x84222325u; h_hi = 0xcbf29ce4u;                   // FNV-1a-64 offset basis
    uint32_t c0 = a.cfg0[env_local];
    if (c0 >= a.n_configs) { c0 = 0; status |= MIG_ST_BAD_ACTION; }
    set_cfg_tables((int)c0);
    busy_mask = 0; down_mask = 0; fsz = 0; next_done = MIG_INF; next_up = MIG_INF; next_crit = MIG_INF;
    g_k = 0; g_T = 0; g_done = 0; n_accepted = 0;
    look_valid = 0; look_tick = 0; look_work = 0; look_due = 0; look_cls = 0; look_id = 0;
    n_trace = 0; i_script = 0;
    for (int w = H1_DROPS; w < kHeaderWords; ++w) hdr[w] = 0u;      // running totals, drops
    begin_span();
    update_power();
    gen_next();
  }

  __device__ __forceinline__ void save() {
#pragma unroll
    for (int p = 0; p < kSlots; ++p) { hdr[H1_UPAT + p] = F(TW_UPAT + p); hdr[H1_POS + p] = F(TW_POS + p); }
    hdr[H1_T] = (uint32_t)t;
    hdr[H1_PK] = (uint32_t)epoch | ((uint32_t)cfg << 8) | ((uint32_t)algo << 16) | (status << 24);
    hdr[H1_NSYS] = n_sys; hdr[H1_HLO] = h_lo; hdr[H1_HHI] = h_hi;
    hdr[H1_GK] = g_k; hdr[H1_GT_LO] = (uint32_t)g_T; hdr[H1_GT_HI] = (uint32_t)(g_T >> 32); hdr[H1_GDONE] = g_done;
    hdr[H1_NACC] = n_accepted; hdr[H1_ISCRIPT] = i_script; hdr[H1_MASKS] = busy_mask | (down_mask << 8) | (fsz << 16);
    hdr[H1_LOOKV] = (uint32_t)look_valid; hdr[H1_LOOKTICK] = (uint32_t)look_tick; hdr[H1_LOOKCLS] = look_cls;
    hdr[H1_LOOKWORK] = (uint32_t)look_work; hdr[H1_LOOKDUE] = (uint32_t)look_due; hdr[H1_LOOKID] = look_id;
    const uint32_t ns = min(n_sys, S);
    for (uint32_t i = 0; i < ns; ++i) { const uint2 km = tb[(2 * i) * NT], rdv = tb[(2 * i + 1) * NT]; gtab[i] = make_uint4(km.x, km.y, rdv.x, rdv.y); }
  }

  __device__ __forceinline__ void load() {
    t = (int)hdr[H1_T];
    const uint32_t pk = hdr[H1_PK];
    epoch = pk & 0xFF; algo = (pk >> 16) & 0xFF; status = pk >> 24;
    set_cfg_tables((int)((pk >> 8) & 0xFF));
    n_sys = hdr[H1_NSYS]; h_lo = hdr[H1_HLO]; h_hi = hdr[H1_HHI];
    g_k = hdr[H1_GK]; g_T = (unsigned long long)hdr[H1_GT_LO] | ((unsigned long long)hdr[H1_GT_HI] << 32); g_done = hdr[H1_GDONE];
    n_accepted = hdr[H1_NACC]; i_script = hdr[H1_ISCRIPT];
    busy_mask = hdr[H1_MASKS] & 0x7Fu; down_mask = (hdr[H1_MASKS] >> 8) & 0x7Fu; fsz = hdr[H1_MASKS] >> 16;
    look_valid = (int)hdr[H1_LOOKV]; look_tick = (int)hdr[H1_LOOKTICK]; look_cls = hdr[H1_LOOKCLS];
    look_work = (int)hdr[H1_LOOKWORK]; look_due = (int)hdr[H1_LOOKDUE]; look_id = hdr[H1_LOOKID];
    const uint32_t ns = min(n_sys, S);
    for (uint32_t i = 0; i < ns; ++i) { const uint4 e = gtab[i]; tb[(2 * i) * NT] = make_uint2(e.x, e.y); tb[(2 * i + 1) * NT] = make_uint2(e.z, e.w); }
    int nd = MIG_INF, nu = MIG_INF;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) {
      F(TW_UPAT + p) = hdr[H1_UPAT + p]; F(TW_POS + p) = hdr[H1_POS + p];
      if ((down_mask >> p) & 1u) nu = min(nu, (int)hdr[H1_UPAT + p]);
      if ((busy_mask >> p) & 1u) {                            // running job: t + ceil(rem / v) never drifts
        const uint32_t pos = hdr[H1_POS + p];
        const uint4 sp = speed_of((ld_km(pos).y >> 20) & 15u, size_at(p));
        F(TW_V + p) = sp.x;
        nd = min(nd, t + rd_magic((int)ld_rd(pos).x, sp));
      }
    }
    next_done = nd; next_up = nu;
    n_trace = 0;
    begin_span();
    update_power();
    compute_next_crit();
  }

  // ------------------------------------------------------------------ n_steps decision epochs, one flat loop
  // `li` indexes this launch's env range (explicit actions), `env` the handle's arrays
  __device__ __forceinline__ void run(uint32_t li, uint32_t env) {
    int steps_left = a.n_steps;
    if (steps_left <= 0 || epoch >= a.n_epochs) return;
    const uint32_t out_i = TRACE ? 0u : env;
    bool drain = false, fresh = true;
    long long dE = 0, dT = 0;
    for (int s = 0;;) {
      if (fresh) {                                            // ---- the next decision epoch begins
        fresh = false; drain = false; dE = 0; dT = 0;
        uint32_t action = (uint32_t)cfg;                                            // STATIC: stay
        if (a.policy == MIG_POLICY_TABLE) {                                         // load bucket
          const uint32_t b = n_sys == 0 ? 0u : (n_sys < 8 ? 1u : (n_sys < 64 ? 2u : 3u));
          action = a.table[((size_t)env * a.n_epochs + epoch) * 4 + b];
        } else if (a.actions) {
          action = a.actions[(size_t)li * a.act_stride_env + (size_t)s * a.act_stride_k];
        }
        begin_span();
        prologue(action);
        t_end = (epoch + 1) * a.epoch_s;
      }
      if (t != t_end && !(drain && n_sys == 0)) { event(); continue; }
      // ---- the span is over
      dE += e_ep; dT += tard_ep;
      if (!drain) {
        hdr[H1_DROPS] = F(TW_CNT + C_DROPPED);
        close_record(a.recs ? a.recs + (size_t)(epoch - a.rec_k0) * a.rec_stride + out_i : nullptr);
        if (epoch == a.n_epochs - 1) {                        // 4. drain (reading #11): energy stops at the last completion
          drain = true; begin_span(); t_end = a.t_limit_s;
          continue;
        }
      } else {
        if (n_sys > 0) status |= MIG_ST_TRUNCATED;
        close_record(a.drain_rec ? a.drain_rec + out_i : nullptr);
      }
      epoch++;
      if (a.energy_out) a.energy_out[out_i] = dE;
      if (a.tard_out) a.tard_out[out_i] = dT;
      if (a.reward_out)                                       // two fp32 products, one add, negate; no contraction
        a.reward_out[out_i] = -__fadd_rn(__fmul_rn(a.w_energy, __ll2float_rn(dE)), __fmul_rn(a.w_tardy, __ll2float_rn(dT)));
      ++s;
      if (--steps_left == 0 || epoch >= a.n_epochs) break;
      fresh = true;
    }
  }
};

template <int NT, bool TRACE>
__global__ void __launch_bounds__(NT) sim_thread_kernel(const SimArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HotTablesT &hot = *reinterpret_cast<HotTablesT *>(smem_raw);
  {
    const DevTables *tb = a.tab;
    for (int i = threadIdx.x; i < MIG_MAX_CLASSES * 5; i += NT) hot.h.speed[i] = tb->speed[i];
    for (int i = threadIdx.x; i < MIG_MAX_CONFIGS; i += NT) {
      hot.h.cfg_pack[i] = tb->cfg_pack[i]; hot.cfg_rank[i] = tb->cfg_rank[i]; hot.cfg_slot_of[i] = tb->cfg_slot_of[i]; hot.cfg_pidle[i] = tb->cfg_pidle[i];
    }
    if (threadIdx.x < 8) { hot.h.curve[threadIdx.x] = tb->curve[threadIdx.x]; hot.h.p_idle[threadIdx.x] = tb->p_idle[threadIdx.x]; hot.h.p_busy[threadIdx.x] = tb->p_busy[threadIdx.x]; }
    for (int i = threadIdx.x; i < 257; i += NT) hot.logT[i] = tb->logT[i];
  }
  __syncthreads();
  const uint32_t li = blockIdx.x * NT + threadIdx.x;            // index inside this launch's env range
  if (li >= a.n_envs) return;
  uint32_t *fx = reinterpret_cast<uint32_t *>(smem_raw + ((sizeof(HotTablesT) + 127) & ~(size_t)127)) + threadIdx.x;
  uint2 *tbl = reinterpret_cast<uint2 *>(fx - threadIdx.x + TW_FIXED * NT) + threadIdx.x;
  EnvT<NT, TRACE> e(a, hot, fx, tbl);
  const uint32_t env = a.env_first + li;
  e.env_g = a.env_base + env;
  e.gtab = a.tab_override ? a.tab_override : a.jobtab + (size_t)env * a.cap;
  e.hdr = a.hdr_override ? a.hdr_override : a.hdr + (size_t)env * kHeaderWords;
  if (a.from_init) e.init(env); else e.load();
  e.run(li, env);
  if (a.state_out) e.observe(a.state_out + (size_t)(TRACE ? 0u : env) * MIG_STATE_DIM);
  if (a.totals) e.store_totals(a.totals + (TRACE ? 0u : env));   // totals so far (hash and t are live values)
  if (a.save) e.save();
  if (TRACE && a.trace_n) *a.trace_n = e.n_trace;
}

}  // namespace migsim
