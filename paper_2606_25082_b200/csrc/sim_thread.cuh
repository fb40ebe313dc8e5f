// sim_thread.cuh -- the rollout kernel with ONE THREAD PER ENVIRONMENT (the library default; mig_sim_set_tile(s, 1)).
//
// Why: the warp-tile kernel of sim_device.cuh spends most of its issue slots on cross-lane plumbing (butterfly
// reductions, ballots, broadcasts) for queues that hold about a dozen jobs and a GPU that has 7 slots.  With one
// environment per lane there is NO cross-lane traffic at all: every lane runs the serial event loop of DESIGN.md 3.3 on
// its own environment and a warp instruction advances up to 32 environments at once; the price is branch divergence
// between lanes, which the hardware reconverges (profiles/ has the measured threads-per-instruction).  One resident
// wave is 148 SMs x 448 threads = 66 304 environments (BASELINE C5: 65 536); smaller batches put fewer environments in
// each warp (SimArgs::envs_per_warp) so that they still spread over the whole machine.
//
// Data structures are chosen so that no step scans the queue (a lane with a 300-job queue would otherwise hold its 31
// neighbours for the length of its scan) and that lanes doing the same thing run the same instructions:
//   * RUNNING jobs live in the slice table: slot p holds {skey, meta, rem, due} and the speed of the job running there;
//   * WAITING jobs live in a sorted two-level double-ended queue on (skey, id): a ring in shared memory for the
//     smallest records, a ring in global memory for the rest.  The reschedule's "all jobs in priority order"
//      is a merge of the <= 7 running jobs with the queue's front; arrivals are inserted from the tail,
//     re-queued jobs from the front (deadlines grow with arrival time, so both are O(1) in practice);
//   * ARRIVALS are drawn before the event loop starts, by gen_arrivals_kernel (gen_kernel.cuh: one warp per environment,
//     32 thinning candidates per pass), into a per-environment list of 8-byte records in global memory (the arrival
//     process does not depend on the schedule); the event loop copies four records at a time into a
//     shared-memory landing slot with cp.async, one block ahead.
// Per-thread data is in shared memory, interleaved by thread (row r of thread tid at base[r * NT + tid]: every access
// of a warp is bank-conflict-free whatever index each lane uses).  Scalars (time, hash, energy, generator, look-ahead
// arrival) live in registers.  The results are bit-identical to the tile kernels and to the oracle
// (tests/test_gpu_parity.py); no code is shared with oracle/.
#pragma once
#include "gen_kernel.cuh"
#include "sim_device.cuh"

namespace migsim {

constexpr int kThreadCta = 64;        // threads (= environments) per CTA of the thread-per-environment kernel
constexpr int kThreadTabExtra = 32;   // job-table entries per env beyond the global ring: save area of the shared ring (16) and the slice table (7)

// per-thread rows of 8 bytes (uint2): slice records, pick staging, then the queue's shared ring; rows of 4 bytes follow
enum { T2_SLKM = 0 /* 7: {skey, meta} of the job running on slot p */, T2_SLRD = 7 /* 7: {rem, due}; a DOWN slice keeps up_at in .x */,
       T2_STG = 14 /* 7: {meta | slot | moved << 3, rem} of pick k */, T2_RING = 21 };
enum { T1_V = 0 /* 7: speed of the running job */, T1_STGDUE = 7 /* 7 */, T1_CNT = 14 /* C_COUNT = 10 */, T1_WORDS = 24 };

// saved per-env header of this kernel (kHeaderWords words); the running totals H1_TOT / H1_CNT live here all the time
enum { H1_T = 0, H1_PK, H1_NSYS, H1_NWAIT, H1_HLO, H1_HHI, H1_GK, H1_GT_LO, H1_GT_HI, H1_GDONE, H1_NACC, H1_ISCRIPT,
       H1_DROPS, H1_MASKS /* busy | down << 8 */, H1_ORDER, H1_QHEAD, H1_QNS, H1_GHEAD, H1_QNG, H1_TOT = 20 /* 6 */, H1_LOOKV = 26, H1_LOOKTICK, H1_LOOKCLS, H1_LOOKWORK,
       H1_LOOKDUE, H1_LOOKID, H1_ACOUNT = 32, H1_AMORE, H1_AID0 /* written by gen_arrivals_kernel */,
       H1_RET = 36 /* discounted return so far, fp32 bits */, H1_DISC /* gamma^k, fp32 bits */, H1_UTIL = 40 /* 8: seconds per utilisation level */,
       H1_CNT = 48 /* 10 */ };
static_assert((int)H1_PK == (int)HG_PK && (int)H1_GK == (int)HG_GK && (int)H1_NACC == (int)HG_NACC && (int)H1_ACOUNT == (int)HG_ACOUNT && (int)H1_AID0 == (int)HG_AID0, "header layout shared with gen_kernel.cuh");

constexpr int kSpeedCols = 6;    // speed columns of this kernel's table: 1g, 2g, 3g, 4g, 7g, MIG disabled (size code 8)
struct HotTablesT {              // per CTA, shared memory
  uint4 speed[MIG_MAX_CLASSES * kSpeedCols];   // {v, magic, shift, 0}
  uint32_t cfg_pack[MIG_MAX_CONFIGS];     // nibble p: size of the slice starting at slot p
  uint32_t cfg_rank[MIG_MAX_CONFIGS];     // nibble p: rank of the slice starting at slot p in (size, slot) order (reading #4)
  uint32_t cfg_slot_of[MIG_MAX_CONFIGS];  // nibble r: start slot of the slice of rank r
  int32_t cfg_pidle[MIG_MAX_CONFIGS];     // sum of p_idle over the slices of the configuration
  int32_t curve[8];
  int32_t pdiff[12];                      // p_busy - p_idle by slice size (0..8)
};
// column of a slice size: 1, 2, 3, 4, 7, 8 -> 0..5;   compute units of a slice: the MIG-disabled GPU (8) has 7
__device__ __forceinline__ int sidx6_of(int size) { return size >= 7 ? size - 3 : size - 1; }
__device__ __forceinline__ int units_of(int size) { return min(size, 7); }

__host__ __device__ constexpr size_t thread_smem_bytes(uint32_t smem_entries, int nt) {
  return ((sizeof(HotTablesT) + 127) & ~(size_t)127) + (size_t)nt * ((T2_RING + 2 * (size_t)smem_entries) * 8 + T1_WORDS * 4 + 32);   // + a 32-byte landing slot: four arrival records
}

// The one-at-a-time arrival generator: draws thinning candidates from (g_k, g_T) until one is accepted or the day ends
// (R2-R5; tables from global memory).  A free function with everything passed and returned BY VALUE and not
// inlined: it is off the hot path, must not cost the event loop registers, and must not make the environment's state
// addressable (a non-inlined member function would pin the whole EnvT in local memory).
struct InlineDraw { uint32_t g_k; unsigned long long g_T; uint32_t done, found, tick, cls, dur7, slack; };
static __device__ __noinline__ InlineDraw draw_next_arrival(const DevTables *tb, uint32_t env_g, uint32_t episode, uint32_t k0, uint32_t k1,
                                                            unsigned long long gap_scale, int day_s, uint32_t g_k, unsigned long long g_T) {
  InlineDraw d; d.done = 0; d.found = 0; d.tick = 0; d.cls = 0; d.dur7 = 0; d.slack = 0;
  uint4 w; unsigned long long tick; uint32_t k;
  for (;;) {
    k = g_k++;
    w = philox4x32_10(k, 0u, env_g, episode, k0, k1);                          // stream 0: gap, accept, class, slack
    g_T += ((unsigned long long)neglog2_q24_tab(w.x, tb->logT) * gap_scale) >> 24;
    tick = g_T >> 16;
    if (tick >= (unsigned long long)day_s) { d.done = 1; break; }               // arrivals stop at the end of the day
    if (w.y <= __ldg(&tb->thr[(uint32_t)tick / 60u])) { d.found = 1; break; }   // Lewis-Shedler thinning
  }
  d.g_k = g_k; d.g_T = g_T;
  if (d.found) {
    const uint32_t c = class_of(w.z, tb->class_cum);                            // (padded with 0xFFFFFFFF beyond n_classes)
    const uint4 wd = philox4x32_10(k, 1u, env_g, episode, k0, k1);              // stream 1: duration
    const uint32_t qi = wd.x >> 26, f = (wd.x >> 16) & 0x3FFu;
    const int q0 = __ldg(&tb->dur7_q[c * 65 + qi]), q1 = __ldg(&tb->dur7_q[c * 65 + qi + 1]);
    d.dur7 = (uint32_t)(q0 + (int)(((long long)(q1 - q0) * (long long)f) >> 10));
    d.slack = __ldg(&tb->slack_lo[c]) + __umulhi(w.w, __ldg(&tb->slack_span[c]));
    d.tick = (uint32_t)tick; d.cls = c;
  }
  return d;
}

// EVD: event-driven decisions of the tabulated policy compiled in (reading #27).  EDF: every environment of the batch runs
// a deadline-keyed algorithm -- EDF-FS, EDF-SS or EDF-SS with restricted preemption (the kernel reads the handle's algorithm
// mask): laxity keys and critical-laxity events are compiled out of this instantiation -- the same results from a shorter
// instruction stream.
template <int NT, bool TRACE, bool EVD, bool EDF>
struct EnvT {
  // ------------------------------------------------------------------ environment state
  const SimArgs &a;
  const HotTablesT &hot;
  uint2 *const r2;         // 8-byte rows: r2[row * NT]
  uint32_t *const r1;      // 4-byte rows: r1[row * NT]
  uint4 *gtab;             // global ring of the waiting queue, then the save area of the shared ring and the slice table
  uint32_t *hdr;           // this env's saved header (running totals are kept there)
  const uint32_t S;        // slots of the shared-memory ring
  uint32_t env_g;
  int t, t_end, epoch, cfg, algo; uint32_t status, n_sys, n_wait, cfg_sizes, cfg_rank, slice_mask;
  uint32_t h_lo, h_hi;
  long long e_ep, tard_ep, busy_ep;
  int P, U, next_crit, next_done, next_up, repartitioned;
  uint32_t busy_mask, down_mask;
  uint32_t q_head, q_ns, g_head, q_ng;   // the waiting queue (n_wait = q_ns + q_ng)
  uint32_t run_order;      // nibble k: slot of the k-th running job in (key, id) order at the last reschedule, 0xF = end
  uint32_t g_k, g_done, n_accepted; unsigned long long g_T;
  int look_valid, look_tick, look_work, look_due; uint32_t look_cls, look_id;
  uint32_t n_trace, i_script, n_events;
  uint32_t env_l; bool in_drain;   // env index in the handle's arrays; the drain after the last epoch is running
  const uint2 *arr;        // this env's arrival list, written by gen_arrivals_kernel (NULL: generate inline)
  uint32_t a_head, a_count, a_id0, a_more;
  uint4 *land;             // landing slot of the asynchronous copy of four list records: rows land[0], land[NT] (cp.async)

  __device__ __forceinline__ EnvT(const SimArgs &a_, const HotTablesT &h_, uint2 *r2_, uint32_t *r1_)
      : a(a_), hot(h_), r2(r2_), r1(r1_), S(a_.smem_entries) {}

  __device__ __forceinline__ uint2 &R2(int row) { return r2[row * NT]; }
  __device__ __forceinline__ uint32_t &R1(int row) { return r1[row * NT]; }
  __device__ __forceinline__ void count(int c, uint32_t n) { r1[(T1_CNT + c) * NT] += n; }

  // ------------------------------------------------------------------ the waiting queue
  // A SORTED double-ended queue on (skey, id) in two levels: the q_ns smallest records in a shared-memory ring of S
  // slots (head q_head), the other q_ng in a global-memory ring (head g_head, capacity a.ring_cap, a power of two);
  // invariant: the global part is empty unless the shared ring is full.  Why not a heap: deadlines are arrival time
  // plus a slack, so a new arrival almost always belongs at the TAIL and a re-queued (preempted) job at the FRONT;
  // insertion costs as many moves as jobs are overtaken (typically 0-2), the minimum is popped in O(1), and -- what
  // matters under SIMT -- every lane that inserts or pops in a given event runs the same few instructions, where heap
  // sifts of queue-dependent depth serialised the lanes of a warp (profiles/r1_thread.md).
  __device__ __forceinline__ uint32_t s_phys(uint32_t i) const { const uint32_t p = q_head + i; return p >= S ? p - S : p; }
  __device__ __forceinline__ uint32_t g_phys(uint32_t i) const { return (g_head + i) & (a.ring_cap - 1u); }
  __device__ __forceinline__ uint2 &SK(uint32_t phys) { return r2[(T2_RING + 2 * phys) * NT]; }
  __device__ __forceinline__ uint2 &SR(uint32_t phys) { return r2[(T2_RING + 2 * phys + 1) * NT]; }
  // rare paths (critical-laxity scans, state vector, save): record at LOGICAL index i in (key, id) order
  __device__ __forceinline__ uint2 ld_km(uint32_t i) {
    if (i < q_ns) return SK(s_phys(i));
    const uint4 e = gtab[g_phys(i - q_ns)]; return make_uint2(e.x, e.y);
  }
  __device__ __forceinline__ uint2 ld_rd(uint32_t i) {
    if (i < q_ns) return SR(s_phys(i));
    const uint4 e = gtab[g_phys(i - q_ns)]; return make_uint2(e.z, e.w);
  }
  __device__ __forceinline__ void st_km(uint32_t i, uint2 km) {
    if (i < q_ns) SK(s_phys(i)) = km; else *reinterpret_cast<uint2 *>(&gtab[g_phys(i - q_ns)]) = km;
  }
  // meta word of this kernel's records: id[12:32) | class[8:12) | crit_cnt[4:8) | 4 scratch bits.  With the id on top,
  // (skey, meta) compared as ONE signed 64-bit number is the (key, id) order (ties -> lower id, reading #5; ids are unique).
  static __device__ __forceinline__ uint32_t m_id(uint32_t m) { return m >> 12; }
  static __device__ __forceinline__ uint32_t m_cls(uint32_t m) { return (m >> 8) & 15u; }
  static __device__ __forceinline__ uint32_t m_crit(uint32_t m) { return (m >> 4) & 15u; }
  static __device__ __forceinline__ long long ord(uint2 x) { return (long long)(((unsigned long long)x.x << 32) | x.y); }
  static __device__ __forceinline__ bool before(uint2 x, uint2 y) { return ord(x) < ord(y); }
  // shared ring, room available: place the record, moving the larger ones one slot towards the tail
  __device__ __forceinline__ void s_insert_back(uint2 km, uint2 rd) {
    const long long o = ord(km);
    uint32_t i = q_ns, p = s_phys(i);
    while (i > 0) {
      const uint32_t pp = p ? p - 1 : S - 1;
      const uint2 qk = SK(pp);
      if (o >= ord(qk)) break;
      SK(p) = qk; SR(p) = SR(pp);
      p = pp; --i;
    }
    SK(p) = km; SR(p) = rd;
    q_ns++;
  }
  // shared ring, room available: the head moves down one slot and the smaller records move towards it
  __device__ __forceinline__ void s_insert_front(uint2 km, uint2 rd) {
    const long long o = ord(km);
    q_head = q_head ? q_head - 1 : S - 1;
    uint32_t i = 0, p = q_head;
    while (i < q_ns) {
      const uint32_t pn = p + 1 == S ? 0 : p + 1;
      const uint2 qk = SK(pn);
      if (o <= ord(qk)) break;
      SK(p) = qk; SR(p) = SR(pn);
      p = pn; ++i;
    }
    SK(p) = km; SR(p) = rd;
    q_ns++;
  }
  __device__ __forceinline__ void g_insert_back(uint2 km, uint2 rd) {
    const long long o = ord(km);
    uint32_t i = q_ng;
    while (i > 0) {
      const uint4 e = gtab[g_phys(i - 1)];
      if (o >= ord(make_uint2(e.x, e.y))) break;
      gtab[g_phys(i)] = e;
      --i;
    }
    gtab[g_phys(i)] = make_uint4(km.x, km.y, rd.x, rd.y);
    q_ng++;
  }
  __device__ __forceinline__ void g_insert_front(uint2 km, uint2 rd) {
    const long long o = ord(km);
    g_head = (g_head - 1u) & (a.ring_cap - 1u);
    uint32_t i = 0;
    while (i < q_ng) {
      const uint4 e = gtab[g_phys(i + 1)];
      if (o <= ord(make_uint2(e.x, e.y))) break;
      gtab[g_phys(i)] = e;
      ++i;
    }
    gtab[g_phys(i)] = make_uint4(km.x, km.y, rd.x, rd.y);
    q_ng++;
  }
  // the shared ring is full: its largest record becomes the smallest of the global part
  __device__ __forceinline__ void spill_tail() {
    const uint32_t p = s_phys(S - 1);
    const uint2 km = SK(p), rd = SR(p);
    g_head = (g_head - 1u) & (a.ring_cap - 1u);
    gtab[g_head] = make_uint4(km.x, km.y, rd.x, rd.y);
    q_ng++; q_ns--;
  }
  // a new arrival: searched from the tail
  __device__ __forceinline__ void queue_push_back(uint2 km, uint2 rd) {
    n_wait++;
    if (q_ns == S) {
      if (ord(km) >= ord(SK(s_phys(S - 1)))) { g_insert_back(km, rd); return; }
      spill_tail();
    }
    s_insert_back(km, rd);
  }
  // a job that was running: searched from the front
  __device__ __forceinline__ void queue_push_front(uint2 km, uint2 rd) {
    n_wait++;
    if (q_ns == S) {
      if (ord(km) >= ord(SK(s_phys(S - 1)))) { g_insert_front(km, rd); return; }
      spill_tail();
    }
    s_insert_front(km, rd);
  }
  __device__ __forceinline__ uint2 queue_top_km() { return SK(q_head); }
  __device__ __forceinline__ uint2 queue_top_rd() { return SR(q_head); }
  __device__ __forceinline__ void queue_refill(const uint4 e) {               // e = gtab[g_head], the smallest of the global part: it moves up into the freed slot
    g_head = (g_head + 1u) & (a.ring_cap - 1u);
    q_ng--;
    const uint32_t p = s_phys(q_ns);
    SK(p) = make_uint2(e.x, e.y); SR(p) = make_uint2(e.z, e.w);
    q_ns++;
  }
  __device__ __forceinline__ void queue_pop() {                              // removes the first record
    q_head = q_head + 1 == S ? 0 : q_head + 1;
    q_ns--; n_wait--;
    if (q_ng) queue_refill(gtab[g_head]);
  }
  // after every key changed (LLF / LALF at a repartition): insertion sort over the logical order
  __device__ __forceinline__ void queue_resort() {
    for (uint32_t i = 1; i < n_wait; ++i) {
      const uint2 km = ld_km(i), rd = ld_rd(i);
      const long long o = ord(km);
      uint32_t j = i;
      while (j > 0 && o < ord(ld_km(j - 1))) { st_rec(j, ld_km(j - 1), ld_rd(j - 1)); --j; }
      if (j != i) st_rec(j, km, rd);
    }
  }
  __device__ __forceinline__ void st_rec(uint32_t i, uint2 km, uint2 rd) {
    if (i < q_ns) { const uint32_t p = s_phys(i); SK(p) = km; SR(p) = rd; } else gtab[g_phys(i - q_ns)] = make_uint4(km.x, km.y, rd.x, rd.y);
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
  __device__ __forceinline__ const uint4 &speed_of(uint32_t cls, int size) const { return hot.speed[cls * kSpeedCols + sidx6_of(size)]; }

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
  __device__ __forceinline__ bool is_lax() const { return !EDF && (algo & ~1) == MIG_ALGO_LLF; }      // LLF or LALF
  __device__ __forceinline__ int skey_of(int due, int rem, uint32_t cls) const {
    if (!is_lax()) return due;                                  // EDF: deadline
    return due - rd_cfg(rem, cls, algo == MIG_ALGO_LALF);                 // laxity + t (t is common to all jobs)
  }

  __device__ __forceinline__ void set_cfg_tables(int c) {
    cfg = c; cfg_sizes = hot.cfg_pack[c]; cfg_rank = hot.cfg_rank[c];
    uint32_t m = 0;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) m |= ((cfg_sizes >> (4 * p)) & 15u) ? (1u << p) : 0u;
    slice_mask = m;
  }

  // run_order without the entry of slot p (a job left its slice): the zero-nibble trick on order ^ pppppppp finds it -- the
  // LOWEST flagged nibble is exact, slots are unique in the list and the 0xF end markers never match p <= 6
  static __device__ __forceinline__ uint32_t drop_slot(uint32_t order, int p) {
    const uint32_t x = order ^ (0x11111111u * (uint32_t)p);
    const uint32_t z = (x - 0x11111111u) & ~x & 0x88888888u;
    if (!z) return order;
    const uint32_t sh = (uint32_t)(__ffs((int)z) - 1) & ~3u, lo = (1u << sh) - 1u;
    return (order & lo) | ((order >> 4) & ~lo) | 0xF0000000u;
  }

  // power and busy units from the slice table (a down slice counts idle)
  __device__ __forceinline__ void update_power() {
    int u = 0, pd = 0;
    for (uint32_t m = busy_mask; m; m &= m - 1) {
      const int g = size_at(__ffs((int)m) - 1);
      u += units_of(g); pd += hot.pdiff[g];
    }
    U = u; P = hot.cfg_pidle[cfg] + pd + hot.curve[u & 7];
  }

  // ------------------------------------------------------------------ arrivals (R2-R5)
  __device__ __forceinline__ uint32_t job_limit() const { return a.job_limit ? min(a.job_limit, MIG_MAX_JOBS) : MIG_MAX_JOBS; }

  // start the asynchronous copy of list records [b, b + 4) (one 32-byte sector) into this thread's landing slot
  // (LDGSTS: no register waits for it).  b is a multiple of 4; the list's capacity is one too.
  __device__ __forceinline__ void fetch_block(uint32_t b) {
    const uint32_t dst = (uint32_t)__cvta_generic_to_shared(land);
    asm volatile("cp.async.cg.shared.global [%0], [%2], 16;\n\tcp.async.cg.shared.global [%1], [%3], 16;\n\tcp.async.commit_group;"
                 ::"r"(dst), "r"(dst + (uint32_t)(NT * sizeof(uint4))), "l"(arr + b), "l"(arr + b + 2) : "memory");
  }

  // The one-at-a-time generator (draw_next_arrival below the struct's forward declaration): used when there is no list
  // (debug trace, mig_sim_set_arrival_buffer(0)) and for the rest of a launch whose list filled up.
  __device__ __forceinline__ void gen_next_inline() {
    if (g_done || n_accepted >= job_limit()) return;
    const InlineDraw d = draw_next_arrival(a.tab, env_g, a.episode, a.k0, a.k1, a.gap_scale, a.day_s, g_k, g_T);
    g_k = d.g_k; g_T = d.g_T; g_done = d.done;
    if (d.found) { set_look(d.tick, d.cls, d.dur7, d.slack); look_id = n_accepted++; }
  }

  // work and due date from the drawn attributes (R5): work = dur7 * v7, due = tick + max(1, dur7 * slack >> 10)
  __device__ __forceinline__ void set_look(uint32_t tick, uint32_t cls, uint32_t dur7, uint32_t slack) {
    unsigned long long rel = ((unsigned long long)dur7 * slack) >> 10;
    if (rel < 1) rel = 1;
    look_tick = (int)tick; look_cls = cls; look_work = (int)(dur7 * hot.speed[cls * kSpeedCols + 4].x);
    look_due = (int)((long long)tick + (long long)rel);
    look_valid = 1;
  }

  // advance the look-ahead to the next accepted arrival (or none)
  __device__ __forceinline__ void gen_next() {
    look_valid = 0;
    if (a.script) {                                      // scripted arrivals (tests), kernel-uniform branch
      if (i_script < a.n_script) {
        const mig_job_t s = a.script[i_script];
        look_valid = 1; look_tick = s.arr; look_cls = s.cls; look_due = s.due;
        look_work = (int)((uint32_t)s.dur7 * hot.speed[s.cls * kSpeedCols + 4].x);
        look_id = i_script; n_accepted++; i_script++;
      }
      return;
    }
    if (arr) {                                                                // the launch's pre-generated list
      if (a_head < a_count) {
        const uint32_t j = a_head & 3u;
        if (j == 0u) asm volatile("cp.async.wait_group 0;" ::: "memory");     // requested one block (>= 1 arrival) ago
        const uint2 e = reinterpret_cast<const uint2 *>(land + (j >> 1) * NT)[j & 1u];
        set_look(e.y & 0x1FFFFu, (e.x >> 25) & 15u, e.x & 0x1FFFFFFu, ((e.x >> 29) << 13) | (e.y >> 17));
        look_id = a_id0 + a_head++;
        if ((a_head & 3u) == 0u && a_head < a_count) fetch_block(a_head);
        return;
      }
      if (!a_more) return;                                                    // nothing more inside this launch's horizon
      arr = nullptr;                                                          // the list was too small: one at a time from here
    }
    gen_next_inline();
  }

  // ------------------------------------------------------------------ reschedule
  // critical-laxity events (LLF / LALF): earliest t_crit = skey - theta > t over waiting jobs
  __device__ __forceinline__ void compute_next_crit() {
    int best = MIG_INF;
    if (is_lax())
      for (uint32_t i = 0; i < n_wait; ++i) {
        const uint2 e = ld_km(i);
        const int tc = (int)e.x - a.theta;
        if (m_crit(e.y) < a.crit_max && tc > t) best = min(best, tc);
      }
    next_crit = best;
  }

  // remove the record at logical index i: the records before it move up one slot, then the front is dropped
  __device__ __forceinline__ void queue_remove_at(uint32_t i) {
    for (uint32_t k = i; k > 0; --k) st_rec(k, ld_km(k - 1), ld_rd(k - 1));
    queue_pop();
  }

  // EDF-SS with RESTRICTED preemption (reading #26).  Running jobs keep their slices; the
  // waiting jobs are visited in (due, id) order = queue order: (a) slowest FREE slice on which the job is on time, else
  // (b) slowest OCCUPIED slice on which it is on time among those whose job has a later (due, id): that job is preempted
  // and waits again (it is visited later in the same pass), else (c) fastest free slice, else (d) it waits.
  __device__ __forceinline__ void reschedule_restricted() {
    const uint32_t up = slice_mask & ~down_mask;
    uint32_t free_m = up & ~busy_mask;
    long long maxrun = (long long)0x8000000000000000ll;      // largest (due, id) among the running jobs
    for (uint32_t m = busy_mask; m; m &= m - 1) maxrun = max(maxrun, ord(R2(T2_SLKM + __ffs((int)m) - 1)));
    uint32_t i = 0; int n_start = 0, n_pre = 0;
    while (i < n_wait) {
      const uint2 km = ld_km(i), rdv = ld_rd(i);
      if (free_m == 0u && ord(km) > maxrun) break;            // nobody from here on can start (the queue is sorted)
      const int rem = (int)rdv.x, slack = (int)rdv.y - t;
      const uint32_t cls = m_cls(km.y);
      int ssf = -1, fsf = MIG_INF, sso = -1;
      for (uint32_t m = up; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const int r = rd_magic(rem, speed_of(cls, size_at(p)));
        const int rk = (int)((cfg_rank >> (4 * p)) & 7u);
        if ((free_m >> p) & 1u) {
          fsf = min(fsf, (r << 3) | rk);
          if (r <= slack) ssf = max(ssf, (r << 3) | (7 - rk));
        } else if (r <= slack && before(km, R2(T2_SLKM + p))) sso = max(sso, (r << 3) | (7 - rk));
      }
      int rk; bool evict = false;
      if (ssf >= 0) rk = 7 - (ssf & 7);                                      // (a)
      else if (sso >= 0) { rk = 7 - (sso & 7); evict = true; }                // (b)
      else if (free_m) rk = fsf & 7;                                          // (c)
      else { ++i; continue; }                                                 // (d)
      const int s = (int)((hot.cfg_slot_of[cfg] >> (4 * rk)) & 7u), g = size_at(s);
      if (i) queue_remove_at(i); else queue_pop();
      if (evict) {
        const uint2 vk = R2(T2_SLKM + s), vr = R2(T2_SLRD + s);
        emit(MIG_EV_PREEMPT, s, (uint32_t)g, m_id(vk.y), (int)vr.x);
        queue_push_front(vk, vr);                                            // its key is later than km: index >= i
        ++n_pre;
      }
      emit(MIG_EV_START, s, (uint32_t)g, m_id(km.y), rem);
      R2(T2_SLKM + s) = make_uint2(rdv.y, km.y & ~15u);
      R2(T2_SLRD + s) = rdv;
      R1(T1_V + s) = speed_of(cls, g).x;
      busy_mask |= 1u << s; free_m &= ~(1u << s);
      ++n_start;
      if (evict) { maxrun = (long long)0x8000000000000000ll; for (uint32_t m = busy_mask; m; m &= m - 1) maxrun = max(maxrun, ord(R2(T2_SLKM + __ffs((int)m) - 1))); }
      else maxrun = max(maxrun, ord(make_uint2(rdv.y, km.y & ~15u)));
    }
    if (n_pre) count(C_PREEMPT, (uint32_t)n_pre);
    if (n_start) count(C_START, (uint32_t)n_start);
    int nd = MIG_INF;
    for (uint32_t m = busy_mask; m; m &= m - 1) {              // completion times never drift: t + ceil(rem / v)
      const int p = __ffs((int)m) - 1;
      nd = min(nd, t + rd_magic((int)R2(T2_SLRD + p).x, speed_of(m_cls(R2(T2_SLKM + p).y), size_at(p))));
    }
    next_done = nd; next_crit = MIG_INF;
    update_power();
  }

  // Every job in the system is re-evaluated: in (key, id) order, while an up slice is left, each job picks a slice by its
  // rule.  The order is produced by merging the running jobs (slice table) with the front of the waiting queue.
  __device__ __forceinline__ void reschedule() {
    if (algo == MIG_ALGO_EDF_SS_R) { reschedule_restricted(); return; }
    if (is_lax())                       // the keys of running jobs move with their remaining work
      for (uint32_t m = busy_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const uint2 km = R2(T2_SLKM + p), rdv = R2(T2_SLRD + p);
        R2(T2_SLKM + p).x = (uint32_t)skey_of((int)rdv.y, (int)rdv.x, m_cls(km.y));
      }
    uint32_t avail = slice_mask & ~down_mask;       // every UP slice, occupied or not
    uint32_t rmask = busy_mask;                     // running jobs not picked yet
    uint32_t keep = 0, nb = 0; int K = 0, nd = MIG_INF, u = 0, pd = 0;
    uint32_t moved_mask = 0;
    uint32_t ro = run_order | 0xF0000000u, new_order = 0xFFFFFFFFu;
    uint4 gh = make_uint4(0u, 0u, 0u, 0u); bool gh_valid = q_ng != 0u;      // the global part's head, requested before the pick that may need it
    if (gh_valid) gh = gtab[g_head];
    while (avail != 0u) {
      // --- next job in (key, id) order: the first of the unpicked running jobs, or the front of the queue
      uint2 bkm = make_uint2(0x7FFFFFFFu, 0xFFFFFFFFu); int bp = -1;
      if (!is_lax()) {                    // EDF keys are static: run_order lists exactly the running jobs, still in key order
        const uint32_t rs = ro & 15u;     // (15: none left); both candidate keys are loaded, the choice is two selects
        const uint2 rkm = R2(T2_SLKM + (int)(rs & 7u)), wk = queue_top_km();      // (valid rows even when there is no such job)
        const bool has_r = rs != 15u, has_w = n_wait != 0u;
        if (!has_r && !has_w) break;                                      // nobody left
        const bool from_q = has_w && (!has_r || before(wk, rkm));
        bkm = from_q ? wk : rkm; bp = from_q ? 7 : (int)rs;
      } else {
        for (uint32_t m = rmask; m; m &= m - 1) {
          const int p = __ffs((int)m) - 1;
          const uint2 km = R2(T2_SLKM + p);
          if (bp < 0 || before(km, bkm)) { bkm = km; bp = p; }
        }
        if (n_wait) {
          const uint2 wk = queue_top_km();
          if (bp < 0 || before(wk, bkm)) { bkm = wk; bp = 7; }
        }
        if (bp < 0) break;                                                // nobody left
      }
      uint2 rdv;
      {                                   // take the record from the queue's front or from the slice table: selects, not a branch
        const bool take_q = bp == 7;
        rdv = r2[(take_q ? T2_RING + 2 * (int)q_head + 1 : T2_SLRD + bp) * NT];      // one load, selected row
        const uint32_t qh1 = q_head + 1u == S ? 0u : q_head + 1u;
        q_head = take_q ? qh1 : q_head;
        q_ns -= take_q ? 1u : 0u; n_wait -= take_q ? 1u : 0u;
        rmask &= take_q ? 0xFFFFFFFFu : ~(1u << bp);
        ro = take_q ? ro : ro >> 4;
        if (take_q && q_ng) {                                             // the smallest of the global part moves up
          if (gh_valid) queue_refill(gh); else queue_refill(gtab[g_head]);
          gh_valid = false;
        }
      }
      const int rem = (int)rdv.x, slack = (int)rdv.y - t;
      const uint32_t cls = m_cls(bkm.y);
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
      const int g = size_at(s);
      avail &= ~(1u << s);
      nb |= 1u << s; nd = min(nd, t + (pick >> 3)); u += units_of(g); pd += hot.pdiff[g];
      const bool moved = bp != s;
      if (!moved) keep |= 1u << s;
      moved_mask |= (moved ? 1u : 0u) << K;
      R2(T2_STG + K) = make_uint2((bkm.y & ~15u) | (uint32_t)s | (moved ? 8u : 0u), rdv.x);
      R1(T1_STGDUE + K) = rdv.y;
      new_order = (new_order & ~(15u << (4 * K))) | ((uint32_t)s << (4 * K));
      ++K;
    }
    // --- diff against the previous assignment: PREEMPT ascending old slot, START in priority order
    const uint32_t pm = busy_mask & ~keep;
    if (pm) {
      count(C_PREEMPT, __popc(pm));
      for (uint32_t m = pm; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        emit(MIG_EV_PREEMPT, p, (uint32_t)size_at(p), m_id(R2(T2_SLKM + p).y), (int)R2(T2_SLRD + p).x);
      }
      for (uint32_t m = rmask; m; m &= m - 1) {                           // running jobs that lost their slice wait again
        const int p = __ffs((int)m) - 1;
        queue_push_front(R2(T2_SLKM + p), R2(T2_SLRD + p));
      }
    }
    const int n_start = __popc(moved_mask);
    for (uint32_t mm = moved_mask; mm; mm &= mm - 1) {                    // only the picks that changed slice: no test inside the loop
      const int k = __ffs((int)mm) - 1;
      const uint2 st = R2(T2_STG + k);
      const int s = (int)(st.x & 7u), g = size_at(s);
      const uint32_t meta = st.x & ~15u, due = R1(T1_STGDUE + k);
      emit(MIG_EV_START, s, (uint32_t)g, m_id(meta), (int)st.y);
      R2(T2_SLKM + s) = make_uint2(due, meta);
      R2(T2_SLRD + s) = make_uint2(st.y, due);
      R1(T1_V + s) = speed_of(m_cls(meta), g).x;
    }
    if (n_start) count(C_START, (uint32_t)n_start);
    busy_mask = nb; next_done = nd; run_order = new_order;
    U = u; P = hot.cfg_pidle[cfg] + pd + hot.curve[u & 7];
    compute_next_crit();
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
    if (a.util_hist && dt) hdr[H1_UTIL + U] += (uint32_t)dt;          // time at this utilisation level (Fig. 6)
    t = tn;
    uint32_t done = 0;
    if (dt)
      for (uint32_t m = busy_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const int rem = (int)R2(T2_SLRD + p).x - dt * (int)R1(T1_V + p);
        R2(T2_SLRD + p).x = (uint32_t)rem;
        if (rem <= 0) done |= 1u << p;
      }
    bool happened = false, job_event = done != 0u;
    for (; done; done &= done - 1) {                                  // (i) completions, ascending slot
      const int p = __ffs((int)done) - 1;
      const int tard = max(t - (int)R2(T2_SLRD + p).y, 0);            // l_j = max(c_j - d_j, 0)
      emit(MIG_EV_COMPLETE, p, (uint32_t)size_at(p), m_id(R2(T2_SLKM + p).y), tard);
      tard_ep += tard;
      count(C_COMPLETED, 1u);
      if (tard > 0) count(C_TARDY, 1u);
      busy_mask &= ~(1u << p);
      run_order = drop_slot(run_order, p);
      n_sys--;
      happened = true;
    }
    if (next_up == t) {                                     // (ii) slices coming up, ascending slot
      int nu = MIG_INF;
      for (uint32_t m = down_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        const int up = (int)R2(T2_SLRD + p).x;
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
        queue_push_back(make_uint2((uint32_t)skey_of(look_due, look_work, look_cls), (look_id << 12) | (look_cls << 8)),
                        make_uint2((uint32_t)look_work, (uint32_t)look_due));
        n_sys++;
        if (n_sys > R1(T1_CNT + C_SYSMAX)) R1(T1_CNT + C_SYSMAX) = n_sys;
      }
      emit(drop ? MIG_EV_DROP : MIG_EV_ARRIVE, 0xFF, look_cls, look_id, look_due);
      happened = true; job_event = true;
      gen_next();
    }
    if (!EDF && next_crit == t) {                                     // (iv) critical laxity, ascending id
      int last_id = -1;
      for (;;) {
        uint32_t bid = 0xFFFFFFFFu, bi = 0; uint2 bkm = make_uint2(0u, 0u);
        for (uint32_t i = 0; i < n_wait; ++i) {                       // jobs present before this tick's arrivals (reading #23)
          const uint2 e = ld_km(i);
          const uint32_t id = m_id(e.y);
          const bool q = id < first_new && m_crit(e.y) < a.crit_max && (int)e.x - a.theta == t && (int)id > last_id;
          if (q && id < bid) { bid = id; bi = i; bkm = e; }
        }
        if (bid == 0xFFFFFFFFu) break;
        const uint32_t cc = m_crit(bkm.y) + 1u;
        st_km(bi, make_uint2(bkm.x, (bkm.y & ~(15u << 4)) | (cc << 4)));
        emit(MIG_EV_CRIT, 0xFF, cc, bid, (int)ld_rd(bi).y);
        count(C_CRIT, 1u);
        last_id = (int)bid;
        happened = true;
      }
    }
    // event-driven decision (reading #27): after a tick of the day with an arrival or a
    // completion the tabulated policy is looked up with the load bucket of this moment
    if (EVD && a.ev_decide && job_event && !in_drain) {
      uint32_t action;
      if (a.policy == MIG_POLICY_BINNED) action = a.bin_table[binned_index()];      // the paper's binned 2+2m state (L210)
      else {
        const uint32_t b = n_sys == 0 ? 0u : (n_sys < 8 ? 1u : (n_sys < 64 ? 2u : 3u));
        action = a.table[((size_t)env_l * a.n_epochs + epoch) * 4 + b];
      }
      if (action >= a.n_configs) status |= MIG_ST_BAD_ACTION;
      else if ((int)action != cfg) { repartition(action); return; }   // (it reschedules)
    }
    if (happened) reschedule();                                       // (v)
  }

  // ------------------------------------------------------------------ repartition (readings #13, #14)
  __device__ __forceinline__ void prologue(uint32_t action) {
    repartitioned = 0;
    if (action >= a.n_configs) { status |= MIG_ST_BAD_ACTION; return; }
    if ((int)action == cfg) return;                           // "remain on the current configuration": no cost, no event
    repartition(action);
  }
  // action is a valid configuration other than the current one; ends with ONE reschedule
  __device__ __forceinline__ void repartition(uint32_t action) {
    const uint32_t newsizes = hot.cfg_pack[action];
    uint32_t changed = 0;                                     // slots whose (start, size) differs between the two rows
#pragma unroll
    for (int p = 0; p < kSlots; ++p) changed |= (((cfg_sizes ^ newsizes) >> (4 * p)) & 15u) ? (1u << p) : 0u;
    if (a.all_down) changed = 0x7Fu;                          // the whole GPU goes down (reading #30)
    const uint32_t pm = busy_mask & changed;                  // jobs on destroyed slices go back to waiting
    if (pm) {
      count(C_PREEMPT, __popc(pm));
      for (uint32_t m = pm; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        emit(MIG_EV_PREEMPT, p, (uint32_t)size_at(p), m_id(R2(T2_SLKM + p).y), (int)R2(T2_SLRD + p).x);
      }
      for (uint32_t m = pm; m; m &= m - 1) {                  // (LLF / LALF keys are recomputed below)
        const int p = __ffs((int)m) - 1;
        queue_push_front(R2(T2_SLKM + p), R2(T2_SLRD + p));
      }
      busy_mask &= ~pm;
      uint32_t o = 0xFFFFFFFFu; int k = 0;                    // run_order keeps the jobs that stay, in their order
      for (uint32_t ro = run_order | 0xF0000000u; (ro & 15u) != 15u; ro >>= 4)
        if ((busy_mask >> (ro & 15u)) & 1u) { o = (o & ~(15u << (4 * k))) | ((ro & 15u) << (4 * k)); ++k; }
      run_order = o;
    }
    const int old = cfg;
    set_cfg_tables((int)action);
    down_mask &= ~changed;                                    // same (start, size) in both rows keeps job and up_at
    if (a.downtime_s > 0)
      for (uint32_t m = changed & slice_mask; m; m &= m - 1) {
        const int p = __ffs((int)m) - 1;
        R2(T2_SLRD + p).x = (uint32_t)(t + a.downtime_s);
        down_mask |= 1u << p;
      }
    int nu = MIG_INF;
    for (uint32_t m = down_mask; m; m &= m - 1) nu = min(nu, (int)R2(T2_SLRD + __ffs((int)m) - 1).x);
    next_up = nu;
    e_ep += a.repart_energy; repartitioned = 1;
    count(C_REPART, 1u);
    emit(MIG_EV_REPART, 0xFF, ((uint32_t)old << 8) | action, MIG_NOJOB, 0);
    if (is_lax() && n_wait) {                     // laxity keys are measured against the configuration: re-key, re-sort
      for (uint32_t i = 0; i < n_wait; ++i) {
        const uint2 km = ld_km(i), rdv = ld_rd(i);
        st_km(i, make_uint2((uint32_t)skey_of((int)rdv.y, (int)rdv.x, m_cls(km.y)), km.y));
      }
      queue_resort();
    }
    reschedule();
  }

  // ------------------------------------------------------------------ records
  __device__ __forceinline__ void begin_span() {
    e_ep = 0; tard_ep = 0; busy_ep = 0; n_events = 0;
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) R1(T1_CNT + i) = (i == C_SYSMAX) ? n_sys : 0u;
    repartitioned = 0;
  }

  // fold the span into the running totals (kept in the env's header); optionally store the 64-byte record
  __device__ __forceinline__ void close_record(mig_epoch_rec_t *r) {
    uint32_t c[C_COUNT];
#pragma unroll
    for (int i = 0; i < C_COUNT; ++i) c[i] = R1(T1_CNT + i);
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
  // job j of the system, running ones first: j < 7 = slot j (valid if busy), j >= 7 = queue record j - 7
  __device__ __forceinline__ bool job_at(uint32_t j, uint2 &km, uint2 &rd) {
    if (j < 7u) { if (!((busy_mask >> j) & 1u)) return false; km = R2(T2_SLKM + (int)j); rd = R2(T2_SLRD + (int)j); return true; }
    km = ld_km(j - 7u); rd = ld_rd(j - 7u); return true;
  }
  __device__ __forceinline__ void observe(float *out) {
    float4 *o4 = reinterpret_cast<float4 *>(out);
#pragma unroll
    for (int w = 0; w < 16; ++w) o4[w] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    for (uint32_t i = 0; i < n_wait; ++i) out[m_cls(ld_km(i).y)] += 1.0f;        // waiting jobs per class (small integers: exact)
    const int n_run = __popc(busy_mask);
    for (uint32_t m = slice_mask; m; m &= m - 1) {
      const int p = __ffs((int)m) - 1, g = size_at(p);
      const float occ = ((down_mask >> p) & 1u) ? 0.5f : (((busy_mask >> p) & 1u) ? 1.0f : 0.0f);
      for (int q = 0; q < units_of(g); ++q) out[16 + p + q] = occ;   // slots covered by this slice
      out[23 + p] = (float)g * 0.125f;
    }
    out[30 + (t / 3600) % 24] = 1.0f;
    out[54] = (float)n_wait * (1.0f / 64.0f);
    out[55] = (float)n_run * 0.125f;
    out[62] = (float)hdr[H1_DROPS] * (1.0f / 64.0f);
    out[63] = 1.0f;
    int pk = (int)0x80000000; uint32_t pid = 0;
    for (int m = 0; m < 3 && (uint32_t)m < n_sys; ++m) {        // first m = 3 jobs in (due, id) order
      uint2 bkm, brd;
      next_by_due(pk, pid, bkm, brd);
      const int d = max(-32768, min(32767, (int)brd.y - t));
      const int mean = min(rd_cfg((int)brd.x, m_cls(bkm.y), true), 32767);
      out[56 + m] = (float)d * (1.0f / 4096.0f);
      out[59 + m] = (float)mean * (1.0f / 4096.0f);
    }
  }
  // the job that follows (pk, pid) in (due, id) order over all jobs in system (running and waiting); advances (pk, pid)
  __device__ __forceinline__ void next_by_due(int &pk, uint32_t &pid, uint2 &bkm, uint2 &brd) {
    int bk = MIG_INF; uint32_t bid = 0xFFFFFFFFu; bkm = make_uint2(0u, 0u); brd = bkm;
    for (uint32_t j = 0; j < 7u + n_wait; ++j) {
      uint2 km, rdv;
      if (!job_at(j, km, rdv)) continue;
      const int due = (int)rdv.y; const uint32_t id = m_id(km.y);
      const bool beyond = due > pk || (due == pk && id > pid);
      const bool better = due < bk || (due == bk && id < bid);
      if (beyond && better) { bk = due; bid = id; bkm = km; brd = rdv; }
    }
    pk = bk; pid = bid;
  }

  // ------------------------------------------------------------------ binned state (reading #31)
  // index of the present state in the BINNED policy's table: configuration, time bin, and for each of the first m = 3 jobs
  // in (due, id) order the code 0 (no such job) or 1 + dbin * n_abins + abin of its deadline (due - t) and its mean
  // remaining duration over the slices of the configuration
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
    for (uint32_t m = 0; m < 3u; ++m) {
      uint32_t code = 0;
      if (m < n_sys) {
        uint2 bkm, brd;
        next_by_due(pk, pid, bkm, brd);
        const uint32_t db = bin_of((int)brd.y - t, a.tab->dbin_edges, a.n_dbins);
        const uint32_t ab = bin_of(rd_cfg((int)brd.x, m_cls(bkm.y), true), a.tab->abin_edges, a.n_abins);
        code = 1u + db * a.n_abins + ab;
      }
      idx = idx * B + code;
    }
    return idx;
  }

  // ------------------------------------------------------------------ init / load / save
  __device__ __forceinline__ void init_regs(uint32_t env_local) {
    algo = a.algo[env_local]; t = 0; epoch = 0; status = 0; n_sys = 0; n_wait = 0;
    if (algo > MIG_ALGO_EDF_SS_R) { algo = MIG_ALGO_EDF_FS; status |= MIG_ST_BAD_ALGO; }   // reading #28
    if (a.algo_mask) {                                        // which algorithms this batch runs (picks the kernel body of later launches)
      const uint32_t act = __activemask(), m = __reduce_or_sync(act, 1u << algo);
      if ((threadIdx.x & 31u) == (uint32_t)(__ffs((int)act) - 1)) atomicOr(a.algo_mask, m);
    }
    q_head = 0; q_ns = 0; g_head = 0; q_ng = 0;
    h_lo = 0x84222325u; h_hi = 0xcbf29ce4u;                   // FNV-1a-64 offset basis
    uint32_t c0 = a.cfg0[env_local];
    if (c0 >= a.n_configs) { c0 = 0; status |= MIG_ST_BAD_ACTION; }
    set_cfg_tables((int)c0);
    busy_mask = 0; down_mask = 0; run_order = 0xFFFFFFFFu; next_done = MIG_INF; next_up = MIG_INF; next_crit = MIG_INF;
    g_k = 0; g_T = 0; g_done = 0; n_accepted = 0; a_count = 0; a_more = 1; a_id0 = 0;
    look_valid = 0; look_tick = 0; look_work = 0; look_due = 0; look_cls = 0; look_id = 0;
    n_trace = 0; i_script = 0;
    for (int w = H1_DROPS; w < kHeaderWords; ++w) hdr[w] = 0u;      // running totals, drops, return, utilisation levels
    hdr[H1_DISC] = __float_as_uint(1.0f);
  }
  __device__ __forceinline__ void init_rows() {
    begin_span();
    update_power();
  }

  __device__ __forceinline__ void save() {
    hdr[H1_T] = (uint32_t)t;
    hdr[H1_PK] = (uint32_t)epoch | ((uint32_t)cfg << 8) | ((uint32_t)algo << 16) | (status << 24);
    hdr[H1_NSYS] = n_sys; hdr[H1_NWAIT] = n_wait; hdr[H1_HLO] = h_lo; hdr[H1_HHI] = h_hi;
    hdr[H1_QHEAD] = q_head; hdr[H1_QNS] = q_ns; hdr[H1_GHEAD] = g_head; hdr[H1_QNG] = q_ng;
    hdr[H1_GK] = g_k; hdr[H1_GT_LO] = (uint32_t)g_T; hdr[H1_GT_HI] = (uint32_t)(g_T >> 32); hdr[H1_GDONE] = g_done;
    hdr[H1_NACC] = n_accepted; hdr[H1_ISCRIPT] = i_script; hdr[H1_MASKS] = busy_mask | (down_mask << 8); hdr[H1_ORDER] = run_order;
    hdr[H1_LOOKV] = (uint32_t)look_valid; hdr[H1_LOOKTICK] = (uint32_t)look_tick; hdr[H1_LOOKCLS] = look_cls;
    hdr[H1_LOOKWORK] = (uint32_t)look_work; hdr[H1_LOOKDUE] = (uint32_t)look_due; hdr[H1_LOOKID] = look_id;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) { const uint2 km = R2(T2_SLKM + p), rdv = R2(T2_SLRD + p); gtab[a.ring_cap + 16 + p] = make_uint4(km.x, km.y, rdv.x, rdv.y); }
    for (uint32_t p = 0; p < S; ++p) { const uint2 km = SK(p), rdv = SR(p); gtab[a.ring_cap + p] = make_uint4(km.x, km.y, rdv.x, rdv.y); }
  }

  __device__ __forceinline__ void load_regs() {
    t = (int)hdr[H1_T];
    const uint32_t pk = hdr[H1_PK];
    epoch = pk & 0xFF; algo = (pk >> 16) & 0xFF; status = pk >> 24;
    set_cfg_tables((int)((pk >> 8) & 0xFF));
    n_sys = hdr[H1_NSYS]; n_wait = hdr[H1_NWAIT]; h_lo = hdr[H1_HLO]; h_hi = hdr[H1_HHI];
    q_head = hdr[H1_QHEAD]; q_ns = hdr[H1_QNS]; g_head = hdr[H1_GHEAD]; q_ng = hdr[H1_QNG];
    g_k = hdr[H1_GK]; g_T = (unsigned long long)hdr[H1_GT_LO] | ((unsigned long long)hdr[H1_GT_HI] << 32); g_done = hdr[H1_GDONE];
    n_accepted = hdr[H1_NACC]; i_script = hdr[H1_ISCRIPT];
    busy_mask = hdr[H1_MASKS] & 0x7Fu; down_mask = (hdr[H1_MASKS] >> 8) & 0x7Fu; run_order = hdr[H1_ORDER];
    look_valid = (int)hdr[H1_LOOKV]; look_tick = (int)hdr[H1_LOOKTICK]; look_cls = hdr[H1_LOOKCLS];
    look_work = (int)hdr[H1_LOOKWORK]; look_due = (int)hdr[H1_LOOKDUE]; look_id = hdr[H1_LOOKID];
    a_count = hdr[H1_ACOUNT]; a_more = hdr[H1_AMORE]; a_id0 = hdr[H1_AID0];      // this launch's list (gen_arrivals_kernel)
  }
  __device__ __forceinline__ void load_rows() {
    for (uint32_t p = 0; p < S; ++p) { const uint4 e = gtab[a.ring_cap + p]; SK(p) = make_uint2(e.x, e.y); SR(p) = make_uint2(e.z, e.w); }
    int nd = MIG_INF, nu = MIG_INF;
#pragma unroll
    for (int p = 0; p < kSlots; ++p) {
      const uint4 e = gtab[a.ring_cap + 16 + p];
      R2(T2_SLKM + p) = make_uint2(e.x, e.y); R2(T2_SLRD + p) = make_uint2(e.z, e.w);
      if ((down_mask >> p) & 1u) nu = min(nu, (int)e.z);
      if ((busy_mask >> p) & 1u) {                            // running job: t + ceil(rem / v) never drifts
        const uint4 sp = speed_of(m_cls(e.y), size_at(p));
        R1(T1_V + p) = sp.x;
        nd = min(nd, t + rd_magic((int)e.z, sp));
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
    in_drain = false;
    long long dE = 0, dT = 0;
    for (int s = 0;;) {
      if (fresh) {                                  // ---- the next decision epoch begins
        fresh = false; drain = false; in_drain = false; dE = 0; dT = 0;
        uint32_t action = (uint32_t)cfg;                                            // STATIC: stay
        if (a.policy == MIG_POLICY_TABLE) {                                         // load bucket
          const uint32_t b = n_sys == 0 ? 0u : (n_sys < 8 ? 1u : (n_sys < 64 ? 2u : 3u));
          action = a.table[((size_t)env * a.n_epochs + epoch) * 4 + b];
        } else if (a.policy == MIG_POLICY_BINNED) {                                 // binned 2+2m state
          action = a.bin_table[binned_index()];
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
        hdr[H1_DROPS] = R1(T1_CNT + C_DROPPED);
        close_record(a.recs ? a.recs + (size_t)(epoch - a.rec_k0) * a.rec_stride + out_i : nullptr);
        if (epoch == a.n_epochs - 1) {                        // 4. drain (reading #11): energy stops at the last completion
          drain = true; in_drain = true; begin_span(); t_end = a.t_limit_s;
          continue;
        }
      } else {
        if (n_sys > 0) status |= MIG_ST_TRUNCATED;
        close_record(a.drain_rec ? a.drain_rec + out_i : nullptr);
      }
      epoch++;
      if (a.energy_out) a.energy_out[out_i] = dE;
      if (a.tard_out) a.tard_out[out_i] = dT;
      {                                                       // reward: two fp32 products, one add, negate; no contraction
        const float r = -__fadd_rn(__fmul_rn(a.w_energy, __ll2float_rn(dE)), __fmul_rn(a.w_tardy, __ll2float_rn(dT)));
        if (a.reward_out) a.reward_out[out_i] = r;
        const float d = __uint_as_float(hdr[H1_DISC]);          // discounted return (reading #32)
        hdr[H1_RET] = __float_as_uint(__fmaf_rn(d, r, __uint_as_float(hdr[H1_RET])));
        hdr[H1_DISC] = __float_as_uint(__fmul_rn(d, a.gamma));
      }
      ++s;
      if (--steps_left == 0 || epoch >= a.n_epochs) break;
      fresh = true;
    }
  }
};

template <int NT, bool TRACE, bool EVD, bool EDF>
__device__ __forceinline__ void thread_body(const SimArgs &a, const HotTablesT &hot, unsigned char *base, uint32_t li) {
  uint2 *r2 = reinterpret_cast<uint2 *>(base) + threadIdx.x;
  uint32_t *r1 = reinterpret_cast<uint32_t *>(base + (size_t)NT * (T2_RING + 2 * (size_t)a.smem_entries) * 8) + threadIdx.x;
  EnvT<NT, TRACE, EVD, EDF> e(a, hot, r2, r1);
  e.land = reinterpret_cast<uint4 *>(base + (size_t)NT * ((T2_RING + 2 * (size_t)a.smem_entries) * 8 + T1_WORDS * 4)) + threadIdx.x;
  const uint32_t env = a.env_first + li;
  e.env_g = a.env_base + env; e.env_l = env; e.in_drain = false;
  e.gtab = a.tab_override ? a.tab_override : a.jobtab + (size_t)env * (a.ring_cap + kThreadTabExtra);
  e.hdr = a.hdr_override ? a.hdr_override : a.hdr + (size_t)env * kHeaderWords;
  e.arr = (a.arr && !a.script) ? a.arr + (size_t)env * a.arr_cap : nullptr;   // (the host launches gen_arrivals_kernel first)
  e.a_head = 0;
  if (a.from_init) { e.init_regs(env); e.init_rows(); } else { e.load_regs(); e.load_rows(); }
  if (a.n_steps > 0 && e.epoch < a.n_epochs) {
    if (e.arr && e.a_count) e.fetch_block(0);
    if (!e.look_valid) e.gen_next();                            // prime the look-ahead (one may be carried over from the last launch)
  }
  e.run(li, env);
  if (a.state_out) e.observe(a.state_out + (size_t)(TRACE ? 0u : env) * MIG_STATE_DIM);
  if (a.totals) e.store_totals(a.totals + (TRACE ? 0u : env));   // totals so far (hash and t are live values)
  if (a.save) e.save();
  if (TRACE && a.trace_n) *a.trace_n = e.n_trace;
}


// The tail of a full-day launch (mig_sim_set_prefetch): a warp whose 32 environments have finished their day draws arrival
// lists of the NEXT episode, one claimed environment at a time, until every warp of the launch has finished its day -- the
// idle lanes of a launch whose warps end between 60 and 69 ms do the generator's work of the next step (the arrival
// process does not depend on the schedule).  What is left is drawn by the next step's gen_arrivals_kernel,
// which skips the flagged environments.  Not inlined and everything BY VALUE: off the hot path, and the kernel's argument
// block must not become addressable.  `mine`: this warp's half of the per-thread rows (dead by now), 256 bytes in every
// 8-byte row = sixteen 16-byte entries; the warp's 128 pending candidates take the first eight rows.
// index of this warp's scheduler in PrefetchArgs::busy: SM id x 4 + warp slot & 3 (a heuristic: only pacing depends on it)
static __device__ __forceinline__ uint32_t sched_slot() {
  uint32_t sm, w;
  asm volatile("mov.u32 %0, %%smid;\n\tmov.u32 %1, %%warpid;" : "=r"(sm), "=r"(w));
  return (sm & 1023u) * 4u + (w & 3u);
}

template <int NT>
static __device__ __noinline__ void tail_prefetch(const PrefetchArgs pf, unsigned char *mine, uint32_t lane) {
  unsigned int *const busy = pf.busy + sched_slot();
  if (lane == 0) { atomicAdd(pf.finished, 1u); atomicSub(busy, 1u); }
  const uint32_t pace_ns = pf.pace_ns;
  const DevTables *t = pf.g.tab;
  const GenTabs tb{t->thr, t->dur7_q, t->class_cum, t->slack_lo, t->slack_span, t->logT};
  for (;;) {
    uint32_t w = 0xFFFFFFFFu;
    if (lane == 0 && *reinterpret_cast<volatile unsigned int *>(pf.finished) < pf.n_warps) w = atomicAdd(pf.claim, 1u);
    w = __shfl_sync(0xffffffffu, w, 0);
    if (w >= pf.g.n_envs) break;                                  // every day of the launch is over, or nothing is left to draw
    uint32_t *o = pf.words + (size_t)w * kGenWords;
    gen_env(pf.g, tb, [mine](uint32_t i) -> GenPend & { return *reinterpret_cast<GenPend *>(mine + (size_t)(i >> 4) * (NT * 8) + (i & 15u) * 16u); },
            [busy, pace_ns] { if (pace_ns && *reinterpret_cast<volatile unsigned int *>(busy)) __nanosleep(pace_ns); },
            lane, pf.g.env_base + w, pf.g.arr + (size_t)w * pf.g.arr_cap, 0, 0u, 0u, 0u, 0ull, o, o + 5);
    __syncwarp();
    if (lane == 0) { __threadfence(); pf.flag[w] = pf.tag; }
  }
}

template <int NT, bool TRACE, bool EVD>
__global__ void __launch_bounds__(NT, 7) sim_thread_kernel(const SimArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HotTablesT &hot = *reinterpret_cast<HotTablesT *>(smem_raw);
  {
    const DevTables *tb = a.tab;
    for (int i = threadIdx.x; i < MIG_MAX_CLASSES * kSpeedCols; i += NT) {
      const int c = i / kSpeedCols, k = i - c * kSpeedCols;
      hot.speed[i] = k < 5 ? tb->speed[c * 5 + k] : tb->speed_nomig[c];
    }
    for (int i = threadIdx.x; i < MIG_MAX_CONFIGS; i += NT) {
      hot.cfg_pack[i] = tb->cfg_pack[i]; hot.cfg_rank[i] = tb->cfg_rank[i]; hot.cfg_slot_of[i] = tb->cfg_slot_of[i]; hot.cfg_pidle[i] = tb->cfg_pidle[i];
    }
    if (threadIdx.x < 8) hot.curve[threadIdx.x] = tb->curve[threadIdx.x];
    if (threadIdx.x < 12) hot.pdiff[threadIdx.x] = tb->p_busy[threadIdx.x] - tb->p_idle[threadIdx.x];
  }
  unsigned char *base = smem_raw + ((sizeof(HotTablesT) + 127) & ~(size_t)127);
  __syncthreads();
  // lanes 0 .. envs_per_warp-1 of every warp hold an environment: small batches are spread over more warps (less
  // divergence per warp, more warps to hide latency); a full batch uses all 32 lanes
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t li = (blockIdx.x * (NT / 32) + (threadIdx.x >> 5)) * a.envs_per_warp + lane;   // index inside this launch's env range
  const bool alive = lane < a.envs_per_warp && li < a.n_envs;
  if (!alive) return;
  const bool tail = a.pf_on && a.envs_per_warp == 32u && li - lane + 31u < a.n_envs;      // a full warp of a full-day launch (warp-uniform)
  if (!TRACE && tail && lane == 0) atomicAdd(a.pf.busy + sched_slot(), 1u);
  // every environment of the batch on EDF-FS / EDF-SS / restricted EDF-SS (bits 0, 1, 4 of the mask that the reset launch
  // collected): the short body
  const bool edf_only = !a.from_init && a.algo_mask && (__ldg(a.algo_mask) & ~0x13u) == 0u;
  if (edf_only) thread_body<NT, TRACE, EVD, true>(a, hot, base, li);
  else thread_body<NT, TRACE, EVD, false>(a, hot, base, li);
  if (!TRACE && tail) {
    __syncwarp();                                               // the warp's 32 days are over: its rows are free
    tail_prefetch<NT>(a.pf, base + (threadIdx.x >> 5) * 256u, lane);
  }
}

// per-env auxiliary results out of the saved headers: the discounted return and the seconds per utilisation level
// (`tiled`: the header was written by the warp-tile kernels, whose layout differs)
__global__ void aux_kernel(const uint32_t *hdr, uint32_t n_envs, int tiled, float *ret_out, int32_t *util_out) {
  const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n_envs) return;
  const uint32_t *h = hdr + (size_t)e * kHeaderWords;
  if (ret_out) ret_out[e] = __uint_as_float(h[tiled ? (int)H_RET : (int)H1_RET]);
  if (util_out) {
    int v[8];
#pragma unroll
    for (int l = 0; l < 8; ++l) v[l] = (int)h[tiled ? tile_util_word(l) : H1_UTIL + l];
    int4 *o = reinterpret_cast<int4 *>(util_out + (size_t)e * 8);
    o[0] = make_int4(v[0], v[1], v[2], v[3]);
    o[1] = make_int4(v[4], v[5], v[6], v[7]);
  }
}

}  // namespace migsim
