/*
 * mig_oracle.c -- CPU ORACLE (test infrastructure only; see mig_oracle.h).
 *
 * One environment = one MIG-partitioned GPU over one simulated day ("queues simulated
 * over 24 hours").  Everything is integer: seconds, milliwatts, int64 millijoules (BASELINE north_star).
 * The code follows DESIGN.md section 3 step by step, in the paper's order and notation:
 *   dur_js  -> rd(j, g) = ceil(rem_j / v[class_j][g])
 *   l_j = max(c_j - d_j, 0)
 *   laxity l_js = d_j - dur_js, measured from the current time (reading #7)
 *   EDF-FS / EDF-SS / LLF / LALF, full re-evaluation at every preemption point (L163)
 *   repartition with a time penalty
 * No blocking, no incremental data structures: linear scans over the jobs in system at every event.
 */
#include "mig_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NONE_JOB 0xFFFFFFFFu
#define NO_SLOT (-1)

static const int SIZE_IDX[8] = { -1, 0, 1, 2, 3, -1, -1, 4 }; /* slice size g -> column of the [..][5] tables */
/* size code 8 = the whole GPU with MIG disabled (reading #29): own speed and power, 7 compute units */
static int units_of(int size) { return size == ORC_SIZE_NOMIG ? 7 : size; }

/* ------------------------------------------------------------------------------------------------
 * R1: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  counter (c0..c3), key (k0,k1); ten rounds,
 * the key bumped by the Weyl constants between rounds. */
void orc_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4])
{
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)M0 * c0;
    uint64_t p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R3: T[i] = round(2^24 log2(1 + i/256)), i = 0..256 */
static uint32_t g_logT[257];
static int g_logT_ready = 0;
static void build_log_table(void)
{
  if (g_logT_ready) return;
  for (int i = 0; i <= 256; ++i) g_logT[i] = (uint32_t)llround(16777216.0 * log2(1.0 + (double)i / 256.0));
  g_logT_ready = 1;
}
void orc_log_table(uint32_t out[257]) { build_log_table(); memcpy(out, g_logT, sizeof(g_logT)); }

static int clz32(uint32_t x) { int n = 0; while (!(x & 0x80000000u)) { x <<= 1; ++n; } return n; } /* x != 0 */

/* R3: E24 = -log2(u) * 2^24 with u = (w|1)/2^32, by table + linear interpolation, all integer */
uint32_t orc_neglog2_q24(uint32_t w)
{
  build_log_table();
  uint32_t m = w | 1u;
  int lz = clz32(m);
  uint32_t y = m << lz;                 /* normalised: top bit set; y/2^31 in [1,2) */
  uint32_t i = (y >> 23) & 0xFFu;
  uint32_t f = (y >> 7) & 0xFFFFu;
  uint32_t L = g_logT[i] + (uint32_t)(((uint64_t)(g_logT[i + 1] - g_logT[i]) * f) >> 16);
  return ((uint32_t)(1 + lz) << 24) - L;
}

uint64_t orc_fnv1a_words(uint64_t h, const uint32_t w[4])
{
  for (int i = 0; i < 4; ++i) { h ^= (uint64_t)w[i]; h *= 0x100000001b3ull; }
  return h;
}

/* ------------------------------------------------------------------------------------------------ */
typedef struct {
  uint32_t id, cls;
  int32_t rem, due;
  uint32_t crit_cnt;
  int slot;        /* start slot of the slice it runs on, or NO_SLOT when waiting */
  int32_t t_crit;  /* absolute time of its next critical-laxity event, or -1 */
} job_t;

typedef struct {
  int size;        /* 0: no slice starts at this slot */
  int down;        /* 1 while being (re)created after a repartition */
  int32_t up_at;
  uint32_t job;    /* id of the job running on it, or NONE_JOB */
} slice_t;

typedef struct { uint32_t n_arrived, n_completed, n_dropped, n_tardy, n_preempt, n_start, n_crit, n_events, n_sys_max;
                 int64_t energy, tard, busy; int repartitioned; } acc_t;

struct orc_env {
  orc_params_t p;
  /* owned copies of the tables */
  uint32_t *speed; int32_t *dur7_q; uint32_t *class_cum; uint16_t *slack_q10; uint8_t *size_at_slot; uint32_t *accept_thr;
  uint32_t *speed_nomig; int32_t *dbin_edges, *abin_edges;
  uint64_t seed; uint32_t env_id, episode;
  /* scripted arrivals */
  orc_job_in_t *script; uint32_t n_script, i_script; int scripted;
  /* generator (R2-R5) */
  uint32_t gen_k; uint64_t gen_Tq16; int gen_done; uint32_t n_accepted;
  struct { int valid; int32_t tick; uint32_t cls; int32_t work, due; uint32_t id; } look;
  /* simulation state */
  int32_t t; int epoch; int cfg; int algo; uint32_t status;
  slice_t sl[ORC_SLOTS];
  job_t *jobs; uint32_t n_sys;     /* jobs in system, kept in arrival (id) order */
  uint64_t hash;
  acc_t ep;                         /* accumulators of the current record span */
  orc_totals_t tot;
  uint32_t last_epoch_drops;
  /* trace */
  orc_event_t *trace; uint32_t trace_cap, n_trace;
  /* event-driven decisions (reading #27): this env's table [n_epochs][4], or NULL */
  const uint8_t *ev_table;
  const uint8_t *bin_table;        /* BINNED policy: the shared table (event-driven look-ups), or NULL */
  int32_t util_s[8];                /* seconds spent with U busy compute units */
};

static void *dup_mem(const void *src, size_t n) { void *d = malloc(n ? n : 1); if (n) memcpy(d, src, n); return d; }

orc_env_t *orc_env_create(const orc_params_t *p, uint64_t seed, uint32_t env_id)
{
  orc_env_t *e = (orc_env_t *)calloc(1, sizeof(*e));
  e->p = *p;
  e->speed = (uint32_t *)dup_mem(p->speed, sizeof(uint32_t) * 5 * p->n_classes);
  e->dur7_q = (int32_t *)dup_mem(p->dur7_q, sizeof(int32_t) * 65 * p->n_classes);
  e->class_cum = (uint32_t *)dup_mem(p->class_cum, sizeof(uint32_t) * p->n_classes);
  e->slack_q10 = (uint16_t *)dup_mem(p->slack_q10, sizeof(uint16_t) * 2 * p->n_classes);
  e->size_at_slot = (uint8_t *)dup_mem(p->size_at_slot, 7 * p->n_configs);
  e->accept_thr = (uint32_t *)dup_mem(p->accept_thr, sizeof(uint32_t) * 1440);
  e->speed_nomig = p->speed_nomig ? (uint32_t *)dup_mem(p->speed_nomig, sizeof(uint32_t) * p->n_classes) : NULL;
  e->dbin_edges = (p->dbin_edges && p->n_dbins > 1) ? (int32_t *)dup_mem(p->dbin_edges, sizeof(int32_t) * (p->n_dbins - 1)) : NULL;
  e->abin_edges = (p->abin_edges && p->n_abins > 1) ? (int32_t *)dup_mem(p->abin_edges, sizeof(int32_t) * (p->n_abins - 1)) : NULL;
  e->seed = seed; e->env_id = env_id;
  e->jobs = (job_t *)calloc(p->cap ? p->cap : 1, sizeof(job_t));
  build_log_table();
  return e;
}

void orc_env_destroy(orc_env_t *e)
{
  if (!e) return;
  free(e->speed); free(e->dur7_q); free(e->class_cum); free(e->slack_q10); free(e->size_at_slot); free(e->accept_thr);
  free(e->speed_nomig); free(e->dbin_edges); free(e->abin_edges);
  free(e->script); free(e->jobs); free(e);
}

void orc_env_set_jobs(orc_env_t *e, const orc_job_in_t *jobs, uint32_t n)
{
  free(e->script);
  e->script = (orc_job_in_t *)dup_mem(jobs, sizeof(orc_job_in_t) * n);
  e->n_script = n; e->scripted = 1;
}

void orc_env_set_trace(orc_env_t *e, orc_event_t *buf, uint32_t cap_events) { e->trace = buf; e->trace_cap = cap_events; e->n_trace = 0; }
uint32_t orc_env_n_events(const orc_env_t *e) { return e->tot.n_events; }
uint32_t orc_env_n_sys(const orc_env_t *e) { return e->n_sys; }

/* ---------------------------------------------------------------------------------------------- events */
static void emit(orc_env_t *e, int type, int slot, uint32_t aux, uint32_t job, int32_t value)
{
  orc_event_t ev;
  ev.t = e->t; ev.type = (uint8_t)type; ev.slot = (uint8_t)(slot < 0 ? 0xFF : slot); ev.aux = (uint16_t)aux;
  ev.job = job; ev.value = value;
  uint32_t w[4] = { (uint32_t)ev.t, (uint32_t)ev.type | ((uint32_t)ev.slot << 8) | ((uint32_t)ev.aux << 16), ev.job,
                    (uint32_t)ev.value };
  e->hash = orc_fnv1a_words(e->hash, w);          /* FNV-1a-64 over the 4 words, emission order */
  if (e->trace && e->n_trace < e->trace_cap) e->trace[e->n_trace] = ev;
  e->n_trace++;
  e->ep.n_events++; e->tot.n_events++;
}

/* ---------------------------------------------------------------------------------------------- generator */
static uint32_t speed_of(const orc_env_t *e, uint32_t cls, int size)
{
  if (size == ORC_SIZE_NOMIG) return e->speed_nomig[cls];          /* MIG disabled: its own column */
  return e->speed[cls * 5 + SIZE_IDX[size]];
}

/* R2-R5: advance to the next accepted arrival (or mark the generator done) */
static void gen_next(orc_env_t *e)
{
  const orc_params_t *p = &e->p;
  e->look.valid = 0;
  if (e->scripted) {
    if (e->i_script < e->n_script) {
      const orc_job_in_t *s = &e->script[e->i_script];
      e->look.valid = 1; e->look.tick = s->arr; e->look.cls = s->cls;
      e->look.work = (int32_t)((uint32_t)s->dur7 * speed_of(e, s->cls, 7)); e->look.due = s->due;
      e->look.id = e->i_script; e->i_script++; e->n_accepted++;
    }
    return;
  }
  uint32_t limit = p->job_limit ? p->job_limit : ORC_MAX_JOBS;
  if (limit > ORC_MAX_JOBS) limit = ORC_MAX_JOBS;
  uint32_t k0 = (uint32_t)e->seed, k1 = (uint32_t)(e->seed >> 32);
  while (!e->gen_done) {
    if (e->n_accepted >= limit) { e->gen_done = 1; break; }
    uint32_t k = e->gen_k;
    uint32_t w[4];
    orc_philox4x32_10(k, 0u, e->env_id, e->episode, k0, k1, w);                 /* stream 0: gap, accept, class, slack */
    uint32_t E24 = orc_neglog2_q24(w[0]);
    uint64_t gap_q16 = ((uint64_t)E24 * p->gap_scale_q16) >> 24;               /* R3: exponential gap, Q16 seconds */
    e->gen_Tq16 += gap_q16;
    uint64_t t = e->gen_Tq16 >> 16;
    if (t >= (uint64_t)p->day_s) { e->gen_done = 1; break; }                   /* arrivals stop at the end of the day */
    e->gen_k = k + 1;
    if (w[1] <= e->accept_thr[t / 60]) {                                       /* R4: Lewis-Shedler thinning */
      uint32_t c = 0;
      while (c + 1 < p->n_classes && w[2] > e->class_cum[c]) ++c;              /* R5: first c with w_class <= cum[c] */
      uint32_t wd[4];
      orc_philox4x32_10(k, 1u, e->env_id, e->episode, k0, k1, wd);              /* stream 1: duration */
      uint32_t i = wd[0] >> 26, f = (wd[0] >> 16) & 0x3FFu;
      const int32_t *q = &e->dur7_q[c * 65];
      int32_t dur7 = q[i] + (int32_t)(((int64_t)(q[i + 1] - q[i]) * (int64_t)f) >> 10);
      uint32_t lo = e->slack_q10[c * 2], hi = e->slack_q10[c * 2 + 1];
      uint32_t slack = lo + (uint32_t)(((uint64_t)w[3] * (uint64_t)(hi - lo + 1)) >> 32);
      uint64_t rel = ((uint64_t)(uint32_t)dur7 * slack) >> 10;
      if (rel < 1) rel = 1;
      e->look.valid = 1; e->look.tick = (int32_t)t; e->look.cls = c;
      e->look.work = (int32_t)((uint32_t)dur7 * speed_of(e, c, 7));
      e->look.due = (int32_t)((int64_t)t + (int64_t)rel);
      e->look.id = e->n_accepted; e->n_accepted++;
      return;
    }
  }
}

/* ---------------------------------------------------------------------------------------------- model */
static int32_t rd(const orc_env_t *e, const job_t *j, int size)   /* remaining duration of j on a slice of that size */
{
  int64_t v = (int64_t)speed_of(e, j->cls, size);
  return (int32_t)(((int64_t)j->rem + v - 1) / v);
}

static job_t *find_job(orc_env_t *e, uint32_t id)
{
  for (uint32_t i = 0; i < e->n_sys; ++i) if (e->jobs[i].id == id) return &e->jobs[i];
  return NULL;
}

/* DESIGN.md 3.1 power: P = curve[U] + sum over slices (busy ? p_busy[g] : p_idle[g]); a down slice is idle */
static void power_now(const orc_env_t *e, int64_t *P, int *U)
{
  int u = 0; int64_t s = 0;
  for (int p = 0; p < ORC_SLOTS; ++p) {
    const slice_t *sl = &e->sl[p];
    if (!sl->size) continue;
    if (sl->size == ORC_SIZE_NOMIG) {
      if (sl->job != NONE_JOB) { u += 7; s += e->p.p_busy_nomig_mw; } else s += e->p.p_idle_nomig_mw;
      continue;
    }
    if (sl->job != NONE_JOB) { u += sl->size; s += e->p.p_busy_mw[SIZE_IDX[sl->size]]; }
    else s += e->p.p_idle_mw[SIZE_IDX[sl->size]];
  }
  *U = u; *P = s + e->p.curve_mw[u];
}

static int n_slices_cfg(const orc_env_t *e) { int n = 0; for (int p = 0; p < ORC_SLOTS; ++p) n += e->sl[p].size != 0; return n; }

/* fastest-slice / mean duration over ALL slices of the current configuration, up or down (readings #7, #8) */
static int32_t rd_fastest_cfg(const orc_env_t *e, const job_t *j)
{
  int32_t best = 0; int have = 0;
  for (int p = 0; p < ORC_SLOTS; ++p) if (e->sl[p].size) { int32_t r = rd(e, j, e->sl[p].size); if (!have || r < best) { best = r; have = 1; } }
  return best;
}
static int32_t rd_mean_cfg(const orc_env_t *e, const job_t *j)
{
  int64_t sum = 0;
  for (int p = 0; p < ORC_SLOTS; ++p) if (e->sl[p].size) sum += rd(e, j, e->sl[p].size);
  return (int32_t)(sum / n_slices_cfg(e));
}

/* priority key, smaller = more urgent */
static int64_t prio_key(const orc_env_t *e, const job_t *j)
{
  switch (e->algo) {
    case ORC_ALGO_LLF:  return (int64_t)j->due - e->t - rd_fastest_cfg(e, j);   /* laxity vs fastest slice of cfg (L179) */
    case ORC_ALGO_LALF: return (int64_t)j->due - e->t - rd_mean_cfg(e, j);      /* laxity vs mean duration over cfg (L183) */
    default:            return (int64_t)j->due;                                  /* EDF (L171-175) */
  }
}

/* slice choice among the still-available slices (avail[p] != 0) */
static int pick_fastest(const orc_env_t *e, const job_t *j, const int *avail)
{
  int best = NO_SLOT; int32_t br = 0;
  for (int p = 0; p < ORC_SLOTS; ++p) {
    if (!avail[p]) continue;
    int32_t r = rd(e, j, e->sl[p].size);
    /* minimise rd; ties -> smaller size, then lower slot (reading #4) */
    if (best == NO_SLOT || r < br || (r == br && e->sl[p].size < e->sl[best].size)) { best = p; br = r; }
  }
  return best;
}
static int pick_slice(const orc_env_t *e, const job_t *j, const int *avail)
{
  if (e->algo == ORC_ALGO_EDF_SS) {           /* slowest slice which can complete it on time, else fastest (L175) */
    int best = NO_SLOT; int32_t br = 0;
    for (int p = 0; p < ORC_SLOTS; ++p) {
      if (!avail[p]) continue;
      int32_t r = rd(e, j, e->sl[p].size);
      if ((int64_t)e->t + r > (int64_t)j->due) continue;
      if (best == NO_SLOT || r > br || (r == br && e->sl[p].size < e->sl[best].size)) { best = p; br = r; }
    }
    if (best != NO_SLOT) return best;
  }
  return pick_fastest(e, j, avail);
}

/* slowest slice of the set `ok` on which j completes by its due date (ties -> smaller size, lower slot), or NO_SLOT */
static int pick_slowest_on_time(const orc_env_t *e, const job_t *j, const int *ok)
{
  int best = NO_SLOT; int32_t br = 0;
  for (int p = 0; p < ORC_SLOTS; ++p) {
    if (!ok[p]) continue;
    int32_t r = rd(e, j, e->sl[p].size);
    if ((int64_t)e->t + r > (int64_t)j->due) continue;
    if (best == NO_SLOT || r > br || (r == br && e->sl[p].size < e->sl[best].size)) { best = p; br = r; }
  }
  return best;
}

/* EDF-SS with RESTRICTED preemption ("a variant that only preempts jobs in cases that directly
 * prevent the jobs from missing their deadlines"; the paper gives no more than this sentence -- the rule below is
 * DESIGN.md reading #26).  Running jobs keep their slices.  The waiting jobs are visited in (due, id) order; job j
 *   (a) takes the slowest FREE up slice on which it finishes on time (the SS rule, L175); otherwise
 *   (b) if it would finish on time on an OCCUPIED up slice whose job has a later (due, id), it takes the slowest such
 *       slice: that job is preempted (PREEMPT, then START of j) and waits again -- it is visited later in this pass;
 *   (c) otherwise, if a free up slice is left, it takes the fastest one (it is late anyway: EDF-SS's fallback, L175);
 *   (d) otherwise it waits.
 * Events are emitted in that order, as they happen. */
static void reschedule_restricted(orc_env_t *e)
{
  uint32_t n = e->n_sys;
  char *seen = (char *)calloc(n ? n : 1, 1);
  for (;;) {
    int best = -1;                            /* jobs[] is in id order: strict '<' keeps the lowest id on ties */
    for (uint32_t i = 0; i < n; ++i) {
      if (e->jobs[i].slot != NO_SLOT || seen[i]) continue;
      if (best < 0 || e->jobs[i].due < e->jobs[best].due) best = (int)i;
    }
    if (best < 0) break;
    seen[best] = 1;
    job_t *j = &e->jobs[best];
    int fr[ORC_SLOTS], oc[ORC_SLOTS], any_free = 0;
    for (int p = 0; p < ORC_SLOTS; ++p) {
      int up = e->sl[p].size && !e->sl[p].down;
      fr[p] = up && e->sl[p].job == NONE_JOB; any_free |= fr[p];
      oc[p] = 0;
      if (up && e->sl[p].job != NONE_JOB) {
        const job_t *r = find_job(e, e->sl[p].job);
        oc[p] = r->due > j->due || (r->due == j->due && r->id > j->id);
      }
    }
    int p = pick_slowest_on_time(e, j, fr);                                   /* (a) */
    if (p == NO_SLOT) {
      p = pick_slowest_on_time(e, j, oc);                                     /* (b) */
      if (p != NO_SLOT) {
        job_t *r = find_job(e, e->sl[p].job);
        emit(e, ORC_EV_PREEMPT, p, (uint32_t)e->sl[p].size, r->id, r->rem); e->ep.n_preempt++; e->tot.n_preempt++;
        r->slot = NO_SLOT; e->sl[p].job = NONE_JOB;
      } else if (any_free) p = pick_fastest(e, j, fr);                        /* (c) */
    }
    if (p == NO_SLOT) continue;                                               /* (d) */
    emit(e, ORC_EV_START, p, (uint32_t)e->sl[p].size, j->id, j->rem); e->ep.n_start++; e->tot.n_start++;
    j->slot = p; e->sl[p].job = j->id;
  }
  for (uint32_t i = 0; i < n; ++i) e->jobs[i].t_crit = -1;
  free(seen);
}

/* "all jobs currently in the system (either actively running ... or waiting in the queue) are
 * re-evaluated for job prioritization and slice allocation.  Any job can be preempted." */
static void reschedule(orc_env_t *e)
{
  if (e->algo == ORC_ALGO_EDF_SS_R) { reschedule_restricted(e); return; }
  uint32_t n = e->n_sys;
  int avail[ORC_SLOTS]; int navail = 0;
  for (int p = 0; p < ORC_SLOTS; ++p) { avail[p] = (e->sl[p].size && !e->sl[p].down); navail += avail[p]; }
  int *newslot = (int *)malloc(sizeof(int) * (n ? n : 1));
  char *taken = (char *)calloc(n ? n : 1, 1);
  uint32_t order[ORC_SLOTS]; int n_order = 0;
  for (uint32_t i = 0; i < n; ++i) newslot[i] = NO_SLOT;
  while (navail > 0) {
    /* next job in (key, id) order: jobs[] is in id order, so a strict '<' keeps the lowest id on ties (reading #5) */
    int best = -1; int64_t bk = 0;
    for (uint32_t i = 0; i < n; ++i) {
      if (taken[i]) continue;
      int64_t k = prio_key(e, &e->jobs[i]);
      if (best < 0 || k < bk) { best = (int)i; bk = k; }
    }
    if (best < 0) break;
    taken[best] = 1;
    int p = pick_slice(e, &e->jobs[best], avail);
    newslot[best] = p; avail[p] = 0; navail--;
    order[n_order++] = (uint32_t)best;
  }
  /* diff against the previous assignment: PREEMPT in ascending old slot, START in priority order */
  for (int p = 0; p < ORC_SLOTS; ++p) {
    if (!e->sl[p].size || e->sl[p].job == NONE_JOB) continue;
    job_t *j = find_job(e, e->sl[p].job);
    uint32_t idx = (uint32_t)(j - e->jobs);
    if (newslot[idx] != p) { emit(e, ORC_EV_PREEMPT, p, (uint32_t)e->sl[p].size, j->id, j->rem); e->ep.n_preempt++; e->tot.n_preempt++; }
  }
  for (int r = 0; r < n_order; ++r) {
    job_t *j = &e->jobs[order[r]];
    int p = newslot[order[r]];
    if (p != j->slot) { emit(e, ORC_EV_START, p, (uint32_t)e->sl[p].size, j->id, j->rem); e->ep.n_start++; e->tot.n_start++; }
  }
  for (int p = 0; p < ORC_SLOTS; ++p) e->sl[p].job = NONE_JOB;
  for (uint32_t i = 0; i < n; ++i) { e->jobs[i].slot = newslot[i]; if (newslot[i] != NO_SLOT) e->sl[newslot[i]].job = e->jobs[i].id; }
  /* critical-laxity events (LLF, LALF only; reading #9): a waiting job's laxity
   * falls by exactly 1 per second, so it reaches the threshold theta at t + (lax - theta). */
  for (uint32_t i = 0; i < n; ++i) {
    job_t *j = &e->jobs[i];
    j->t_crit = -1;
    if ((e->algo == ORC_ALGO_LLF || e->algo == ORC_ALGO_LALF) && j->slot == NO_SLOT && j->crit_cnt < e->p.crit_max) {
      int64_t lax = prio_key(e, j);
      if (lax > (int64_t)e->p.crit_laxity_s) j->t_crit = (int32_t)((int64_t)e->t + (lax - e->p.crit_laxity_s));
    }
  }
  free(newslot); free(taken);
}

static void remove_job(orc_env_t *e, uint32_t idx)
{
  memmove(&e->jobs[idx], &e->jobs[idx + 1], sizeof(job_t) * (e->n_sys - idx - 1));
  e->n_sys--;
}

/* ---------------------------------------------------------------------------------------------- binned state */
/* "2+2m different features: the current MIG configuration, time, and the deadlines and average duration
 * of the first m jobs ... binned", m = 3.  Reading #31: the first m jobs are the first three in (due, id) order over all
 * jobs in system; the deadline feature is due - t, the average duration the mean remaining duration over the slices of
 * the current configuration (as in LALF, L183); a value falls in the first bin i with value < edge[i] (else the last
 * bin); an absent job has code 0, a present one code 1 + dbin * n_abins + abin; time bin = min(t, day_s - 1) * n_tbins
 * / day_s.  index = (((cfg * n_tbins + tbin) * B + code_0) * B + code_1) * B + code_2 with B = 1 + n_dbins * n_abins. */
static uint32_t bin_of(int64_t v, const int32_t *edges, uint32_t n_bins)
{
  uint32_t b = 0;
  while (b + 1 < n_bins && v >= (int64_t)edges[b]) ++b;
  return b;
}
uint32_t orc_env_binned_index(const orc_env_t *e)
{
  const orc_params_t *p = &e->p;
  uint32_t B = 1u + p->n_dbins * p->n_abins;
  int64_t tc = e->t < p->day_s - 1 ? e->t : p->day_s - 1;
  uint32_t tbin = (uint32_t)((tc * (int64_t)p->n_tbins) / p->day_s);
  uint32_t idx = (uint32_t)e->cfg * p->n_tbins + tbin;
  char *taken = (char *)calloc(e->n_sys ? e->n_sys : 1, 1);
  for (int m = 0; m < 3; ++m) {
    int best = -1;                              /* jobs[] is in id order: strict '<' keeps the lowest id on ties */
    for (uint32_t i = 0; i < e->n_sys; ++i) if (!taken[i] && (best < 0 || e->jobs[i].due < e->jobs[best].due)) best = (int)i;
    uint32_t code = 0;
    if (best >= 0) {
      taken[best] = 1;
      uint32_t db = bin_of((int64_t)e->jobs[best].due - e->t, e->dbin_edges, p->n_dbins);
      uint32_t ab = bin_of((int64_t)rd_mean_cfg(e, &e->jobs[best]), e->abin_edges, p->n_abins);
      code = 1u + db * p->n_abins + ab;
    }
    idx = idx * B + code;
  }
  free(taken);
  return idx;
}
void orc_env_util_hist(const orc_env_t *e, int32_t out[8]) { memcpy(out, e->util_s, sizeof(e->util_s)); }

/* ---------------------------------------------------------------------------------------------- event loop */
static void repartition(orc_env_t *e, uint8_t action);

static void run_until(orc_env_t *e, int32_t t_end, int drain)
{
  for (;;) {
    if (drain && e->n_sys == 0) break;                       /* energy stops at the last completion (reading #12) */
    /* 2. next event time */
    int64_t tn = t_end;
    if (e->look.valid && e->look.tick < tn) tn = e->look.tick;
    for (int p = 0; p < ORC_SLOTS; ++p) {
      slice_t *s = &e->sl[p];
      if (!s->size) continue;
      if (s->job != NONE_JOB) { int64_t c = (int64_t)e->t + rd(e, find_job(e, s->job), s->size); if (c < tn) tn = c; }
      if (s->down && s->up_at < tn) tn = s->up_at;
    }
    for (uint32_t i = 0; i < e->n_sys; ++i)
      if (e->jobs[i].slot == NO_SLOT && e->jobs[i].t_crit >= 0 && e->jobs[i].t_crit < tn) tn = e->jobs[i].t_crit;
    int64_t dt = tn - e->t;
    /* integrate power and progress over [t, tn) */
    int64_t P; int U; power_now(e, &P, &U);
    e->ep.energy += P * dt; e->ep.busy += (int64_t)U * dt;
    e->util_s[U] += (int32_t)dt;                                /* time at this utilisation level (Fig. 6) */
    for (int p = 0; p < ORC_SLOTS; ++p) {
      slice_t *s = &e->sl[p];
      if (s->size && s->job != NONE_JOB) { job_t *j = find_job(e, s->job); j->rem -= (int32_t)(dt * (int64_t)speed_of(e, j->cls, s->size)); }
    }
    e->t = (int32_t)tn;
    /* 3. same-tick order (reading #10): completions, slice-ups, arrivals, critical laxity, then ONE reschedule */
    int happened = 0, job_event = 0;
    for (int p = 0; p < ORC_SLOTS; ++p) {                                   /* (i) completions, ascending slot */
      slice_t *s = &e->sl[p];
      if (!s->size || s->job == NONE_JOB) continue;
      job_t *j = find_job(e, s->job);
      if (j->rem > 0) continue;
      int32_t tard = e->t - j->due; if (tard < 0) tard = 0;               /* l_j = max(c_j - d_j, 0) */
      emit(e, ORC_EV_COMPLETE, p, (uint32_t)s->size, j->id, tard);
      e->ep.tard += tard; e->ep.n_completed++; e->tot.n_completed++;
      if (tard > 0) { e->ep.n_tardy++; e->tot.n_tardy++; }
      s->job = NONE_JOB;
      remove_job(e, (uint32_t)(j - e->jobs));
      happened = 1; job_event = 1;
    }
    for (int p = 0; p < ORC_SLOTS; ++p) {                                   /* (ii) slices coming up */
      slice_t *s = &e->sl[p];
      if (s->size && s->down && s->up_at == e->t) { s->down = 0; emit(e, ORC_EV_SLICE_UP, p, (uint32_t)s->size, NONE_JOB, 0); happened = 1; }
    }
    while (e->look.valid && e->look.tick == e->t) {                        /* (iii) arrivals, candidate order */
      e->ep.n_arrived++; e->tot.n_jobs++;
      if (e->n_sys == e->p.cap) {                                          /* queue cap (BASELINE C3/C5) */
        emit(e, ORC_EV_DROP, NO_SLOT, e->look.cls, e->look.id, e->look.due);
        e->ep.n_dropped++; e->tot.n_dropped++;
      } else {
        job_t *j = &e->jobs[e->n_sys++];
        j->id = e->look.id; j->cls = e->look.cls; j->rem = e->look.work; j->due = e->look.due;
        j->crit_cnt = 0; j->slot = NO_SLOT; j->t_crit = -1;
        emit(e, ORC_EV_ARRIVE, NO_SLOT, j->cls, j->id, j->due);
        if (e->n_sys > e->ep.n_sys_max) e->ep.n_sys_max = e->n_sys;
        if (e->n_sys > e->tot.n_sys_max) e->tot.n_sys_max = e->n_sys;
      }
      happened = 1; job_event = 1;
      gen_next(e);
    }
    for (uint32_t i = 0; i < e->n_sys; ++i) {                              /* (iv) critical laxity, ascending id */
      job_t *j = &e->jobs[i];
      if (j->slot == NO_SLOT && j->t_crit == e->t) {
        j->crit_cnt++;
        emit(e, ORC_EV_CRIT, NO_SLOT, j->crit_cnt, j->id, j->due);
        e->ep.n_crit++; e->tot.n_crit++;
        happened = 1;
      }
    }
    /* Event-driven decision ("re-partitioning can happen when a job arrives or is completed"; reading
     * #27): after a tick of the day in which a job arrived or completed, the tabulated policy is looked up again with
     * the load bucket of that moment; a different configuration is a repartition at this very tick (it reschedules). */
    if (job_event && (e->ev_table || e->bin_table) && !drain) {
      uint32_t n = e->n_sys; int b = n == 0 ? 0 : (n < 8 ? 1 : (n < 64 ? 2 : 3));
      uint8_t action = e->bin_table ? e->bin_table[orc_env_binned_index(e)] : e->ev_table[e->epoch * 4 + b];
      if (action >= e->p.n_configs) e->status |= ORC_ST_BAD_ACTION;
      else if ((int)action != e->cfg) { repartition(e, action); happened = 0; }
    }
    if (happened) reschedule(e);                                           /* (v) */
    if (e->t == t_end) break;
  }
}

/* 1. prologue: repartition at the start of an epoch (readings #13, #14) */
static void prologue(orc_env_t *e, uint8_t action)
{
  e->ep.repartitioned = 0;
  if (action >= e->p.n_configs) { e->status |= ORC_ST_BAD_ACTION; return; }
  if ((int)action == e->cfg) return;                      /* "remain on the current configuration": no cost, no event */
  repartition(e, action);
}

/* action is a valid configuration other than the current one */
static void repartition(orc_env_t *e, uint8_t action)
{
  const uint8_t *row = &e->size_at_slot[(uint32_t)action * 7];
  for (int p = 0; p < ORC_SLOTS; ++p) {                   /* destroyed slices, ascending slot: running job goes back to waiting */
    slice_t *s = &e->sl[p];
    if (s->size && (s->size != row[p] || e->p.repart_all_down)) {   /* reading #30: the whole GPU goes down */
      if (s->job != NONE_JOB) {
        job_t *j = find_job(e, s->job);
        emit(e, ORC_EV_PREEMPT, p, (uint32_t)s->size, j->id, j->rem);
        e->ep.n_preempt++; e->tot.n_preempt++;
        j->slot = NO_SLOT; j->t_crit = -1; s->job = NONE_JOB;
      }
    }
  }
  for (int p = 0; p < ORC_SLOTS; ++p) {
    slice_t *s = &e->sl[p];
    if (s->size == row[p] && !e->p.repart_all_down) continue;   /* same (start, size) in both rows: keeps job and up_at */
    s->size = row[p]; s->job = NONE_JOB; s->down = 0; s->up_at = 0;
    if (s->size && e->p.repart_downtime_s > 0) { s->down = 1; s->up_at = e->t + e->p.repart_downtime_s; }
  }
  int old = e->cfg;
  e->cfg = action;
  e->ep.energy += e->p.repart_energy_mj;
  e->ep.repartitioned = 1; e->tot.n_repart++;
  emit(e, ORC_EV_REPART, NO_SLOT, ((uint32_t)old << 8) | action, NONE_JOB, 0);
  reschedule(e);
}

void orc_env_reset(orc_env_t *e, uint32_t episode, uint8_t algo, uint8_t cfg0)
{
  e->episode = episode; e->algo = algo; e->cfg = cfg0;
  e->t = 0; e->epoch = 0; e->status = 0; e->n_sys = 0;
  if (algo > ORC_ALGO_EDF_SS_R) { e->algo = ORC_ALGO_EDF_FS; e->status |= ORC_ST_BAD_ALGO; }   /* reading #28 */
  e->hash = 0xcbf29ce484222325ull;
  memset(&e->ep, 0, sizeof(e->ep)); memset(&e->tot, 0, sizeof(e->tot));
  e->last_epoch_drops = 0; e->n_trace = 0;
  memset(e->util_s, 0, sizeof(e->util_s));
  const uint8_t *row = &e->size_at_slot[(uint32_t)cfg0 * 7];
  for (int p = 0; p < ORC_SLOTS; ++p) { e->sl[p].size = row[p]; e->sl[p].down = 0; e->sl[p].up_at = 0; e->sl[p].job = NONE_JOB; }
  e->gen_k = 0; e->gen_Tq16 = 0; e->gen_done = 0; e->n_accepted = 0; e->i_script = 0;
  gen_next(e);
}

static void close_record(orc_env_t *e, orc_epoch_rec_t *r)
{
  e->tot.energy_mj += e->ep.energy; e->tot.tardiness_s += e->ep.tard; e->tot.busy_unit_s += e->ep.busy;
  e->tot.trace_hash = e->hash; e->tot.t_end = e->t; e->tot.status = e->status;
  if (!r) return;
  memset(r, 0, sizeof(*r));
  r->energy_mj = e->ep.energy; r->tardiness_s = e->ep.tard; r->trace_hash = e->hash;
  r->busy_unit_s = (int32_t)e->ep.busy; r->t_end = e->t; r->n_events = e->ep.n_events;
  r->n_arrived = (uint16_t)e->ep.n_arrived; r->n_completed = (uint16_t)e->ep.n_completed; r->n_dropped = (uint16_t)e->ep.n_dropped;
  r->n_tardy = (uint16_t)e->ep.n_tardy; r->n_preempt = (uint16_t)e->ep.n_preempt; r->n_start = (uint16_t)e->ep.n_start;
  r->n_crit = (uint16_t)e->ep.n_crit; r->n_sys_end = (uint16_t)e->n_sys;
  r->cfg = (uint8_t)e->cfg; r->repartitioned = (uint8_t)e->ep.repartitioned; r->status = (uint8_t)e->status;
  int nr = 0; for (int p = 0; p < ORC_SLOTS; ++p) nr += (e->sl[p].size && e->sl[p].job != NONE_JOB);
  r->n_running_end = (uint8_t)nr; r->n_sys_max = e->ep.n_sys_max;
}

int orc_env_step(orc_env_t *e, uint8_t action, float *state_out, float *reward_out, int64_t *energy_out,
                 int64_t *tardiness_out, orc_epoch_rec_t *rec_out)
{
  if (e->epoch >= e->p.n_epochs) return -1;
  int k = e->epoch;
  memset(&e->ep, 0, sizeof(e->ep)); e->ep.n_sys_max = e->n_sys;
  prologue(e, action);
  run_until(e, (int32_t)(k + 1) * e->p.epoch_s, 0);
  int64_t dE = e->ep.energy, dT = e->ep.tard;
  e->last_epoch_drops = e->ep.n_dropped;
  close_record(e, rec_out ? &rec_out[0] : NULL);
  if (k == e->p.n_epochs - 1) {                        /* 4. drain (reading #11) */
    memset(&e->ep, 0, sizeof(e->ep)); e->ep.n_sys_max = e->n_sys;
    run_until(e, e->p.t_limit_s, 1);
    if (e->n_sys > 0) e->status |= ORC_ST_TRUNCATED;
    dE += e->ep.energy; dT += e->ep.tard;
    close_record(e, rec_out ? &rec_out[1] : NULL);
  }
  e->epoch = k + 1;
  if (energy_out) *energy_out = dE;
  if (tardiness_out) *tardiness_out = dT;
  if (reward_out) {                                     /* two fp32 products, one add, negate; no contraction */
    volatile float a = e->p.w_energy * (float)dE;
    volatile float b = e->p.w_tardy * (float)dT;
    *reward_out = -(a + b);
  }
  if (state_out) orc_env_observe(e, state_out);
  return 0;
}

/* 3.5 state vector: every entry is a small integer times a power of two, exact in fp32 */
void orc_env_observe(const orc_env_t *e, float *x)
{
  for (int i = 0; i < ORC_STATE_DIM; ++i) x[i] = 0.0f;
  uint32_t n_wait = 0, n_run = 0;
  for (uint32_t i = 0; i < e->n_sys; ++i) {
    const job_t *j = &e->jobs[i];
    if (j->slot == NO_SLOT) { x[j->cls] += 1.0f; n_wait++; } else n_run++;
  }
  for (int p = 0; p < ORC_SLOTS; ++p) {
    const slice_t *s = &e->sl[p];
    if (!s->size) continue;
    float v = s->down ? 0.5f : (s->job != NONE_JOB ? 1.0f : 0.0f);
    for (int q = p; q < p + units_of(s->size) && q < ORC_SLOTS; ++q) x[16 + q] = v;
    x[23 + p] = (float)s->size / 8.0f;
  }
  x[30 + (e->t / 3600) % 24] = 1.0f;
  x[54] = (float)n_wait / 64.0f; x[55] = (float)n_run / 8.0f;
  /* deadlines and average duration of the first m = 3 jobs, in (due, id) order */
  char *taken = (char *)calloc(e->n_sys ? e->n_sys : 1, 1);
  for (int m = 0; m < 3; ++m) {
    int best = -1;
    for (uint32_t i = 0; i < e->n_sys; ++i) if (!taken[i] && (best < 0 || e->jobs[i].due < e->jobs[best].due)) best = (int)i;
    if (best < 0) break;
    taken[best] = 1;
    int64_t d = (int64_t)e->jobs[best].due - e->t; if (d < -32768) d = -32768; if (d > 32767) d = 32767;
    x[56 + m] = (float)d / 4096.0f;
    int32_t mean = rd_mean_cfg(e, &e->jobs[best]); if (mean > 32767) mean = 32767;
    x[59 + m] = (float)mean / 4096.0f;
  }
  free(taken);
  x[62] = (float)e->last_epoch_drops / 64.0f; x[63] = 1.0f;
}

void orc_env_totals(const orc_env_t *e, orc_totals_t *out) { *out = e->tot; out->trace_hash = e->hash; out->t_end = e->t; out->status = e->status; }

/* ---------------------------------------------------------------------------------------------- Q-network */
static void q_forward_f32(const orc_qnet_t *q, const float *x, float *h1, float *h2, float *out)
{
  uint32_t H = q->hidden, A = q->n_actions;
  for (uint32_t n = 0; n < H; ++n) { float acc = q->b1[n]; for (uint32_t k = 0; k < ORC_STATE_DIM; ++k) acc = fmaf(x[k], q->W1[k * H + n], acc); h1[n] = acc > 0.0f ? acc : 0.0f; }
  for (uint32_t n = 0; n < H; ++n) { float acc = q->b2[n]; for (uint32_t k = 0; k < H; ++k) acc = fmaf(h1[k], q->W2[k * H + n], acc); h2[n] = acc > 0.0f ? acc : 0.0f; }
  for (uint32_t n = 0; n < A; ++n) { float acc = q->b3[n]; for (uint32_t k = 0; k < H; ++k) acc = fmaf(h2[k], q->W3[k * A + n], acc); out[n] = acc; }
}

static uint8_t argmax_lowest(const float *v, uint32_t n) { uint32_t b = 0; for (uint32_t i = 1; i < n; ++i) if (v[i] > v[b]) b = i; return (uint8_t)b; }

void orc_q_eval(const orc_qnet_t *q, const float *state, uint32_t B, float *q_out, uint8_t *argmax_out)
{
  float *h1 = (float *)malloc(sizeof(float) * q->hidden), *h2 = (float *)malloc(sizeof(float) * q->hidden);
  float *tmp = (float *)malloc(sizeof(float) * q->n_actions);
  for (uint32_t b = 0; b < B; ++b) {
    q_forward_f32(q, state + (size_t)b * ORC_STATE_DIM, h1, h2, tmp);
    if (q_out) memcpy(q_out + (size_t)b * q->n_actions, tmp, sizeof(float) * q->n_actions);
    if (argmax_out) argmax_out[b] = argmax_lowest(tmp, q->n_actions);
  }
  free(h1); free(h2); free(tmp);
}

void orc_q_eval_f64(const orc_qnet_t *q, const float *state, uint32_t B, double *q_out)
{
  uint32_t H = q->hidden, A = q->n_actions;
  double *h1 = (double *)malloc(sizeof(double) * H), *h2 = (double *)malloc(sizeof(double) * H);
  for (uint32_t b = 0; b < B; ++b) {
    const float *x = state + (size_t)b * ORC_STATE_DIM;
    for (uint32_t n = 0; n < H; ++n) { double acc = q->b1[n]; for (uint32_t k = 0; k < ORC_STATE_DIM; ++k) acc += (double)x[k] * (double)q->W1[k * H + n]; h1[n] = acc > 0 ? acc : 0; }
    for (uint32_t n = 0; n < H; ++n) { double acc = q->b2[n]; for (uint32_t k = 0; k < H; ++k) acc += h1[k] * (double)q->W2[k * H + n]; h2[n] = acc > 0 ? acc : 0; }
    for (uint32_t n = 0; n < A; ++n) { double acc = q->b3[n]; for (uint32_t k = 0; k < H; ++k) acc += h2[k] * (double)q->W3[k * A + n]; q_out[(size_t)b * A + n] = acc; }
  }
  free(h1); free(h2);
}

/* ---------------------------------------------------------------------------------------------- whole day */
int orc_rollout(const orc_params_t *p, uint64_t seed, uint32_t env_id, uint32_t episode, uint8_t algo, uint8_t cfg0,
                int policy, const uint8_t *table, const orc_qnet_t *q, float epsilon,
                const orc_job_in_t *jobs, uint32_t n_jobs,
                orc_epoch_rec_t *recs_out, orc_totals_t *totals_out,
                orc_event_t *trace_buf, uint32_t trace_cap, uint32_t *n_trace_out,
                float *states_out, uint8_t *actions_out, float *rewards_out)
{
  return orc_rollout_ex(p, seed, env_id, episode, algo, cfg0, policy, table, q, epsilon, jobs, n_jobs, recs_out, totals_out,
                        trace_buf, trace_cap, n_trace_out, states_out, actions_out, rewards_out, NULL, NULL);
}

int orc_rollout_ex(const orc_params_t *p, uint64_t seed, uint32_t env_id, uint32_t episode, uint8_t algo, uint8_t cfg0,
                   int policy, const uint8_t *table, const orc_qnet_t *q, float epsilon,
                   const orc_job_in_t *jobs, uint32_t n_jobs,
                   orc_epoch_rec_t *recs_out, orc_totals_t *totals_out,
                   orc_event_t *trace_buf, uint32_t trace_cap, uint32_t *n_trace_out,
                   float *states_out, uint8_t *actions_out, float *rewards_out,
                   float *return_out, int32_t *util_out)
{
  orc_env_t *e = orc_env_create(p, seed, env_id);
  if (jobs) orc_env_set_jobs(e, jobs, n_jobs);
  if (trace_buf) orc_env_set_trace(e, trace_buf, trace_cap);
  orc_env_reset(e, episode, algo, cfg0);
  e->ev_table = (policy == ORC_POLICY_TABLE && p->decide_on_events) ? table : NULL;
  e->bin_table = (policy == ORC_POLICY_BINNED && p->decide_on_events) ? table : NULL;
  float G = 0.0f, disc = 1.0f;                                               /* discounted return */
  float x[ORC_STATE_DIM];
  orc_env_observe(e, x);
  double et = (double)epsilon * 4294967296.0;
  uint32_t eps_thr = et >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)llround(et);
  float qv[256];
  orc_epoch_rec_t two[2];
  for (int k = 0; k < p->n_epochs; ++k) {
    if (states_out) memcpy(states_out + (size_t)k * ORC_STATE_DIM, x, sizeof(x));
    uint8_t action = (uint8_t)e->cfg;                                        /* STATIC: stay */
    if (policy == ORC_POLICY_TABLE) {                                        /* DESIGN.md 3.6 load buckets */
      uint32_t n = e->n_sys; int b = n == 0 ? 0 : (n < 8 ? 1 : (n < 64 ? 2 : 3));
      action = table[k * 4 + b];
    } else if (policy == ORC_POLICY_BINNED) {                                /* the paper's binned 2+2m state (L210) */
      action = table[orc_env_binned_index(e)];
    } else if (policy == ORC_POLICY_DQN) {                                   /* eps-greedy */
      uint32_t w[4];
      orc_philox4x32_10((uint32_t)k, 2u, env_id, episode, (uint32_t)seed, (uint32_t)(seed >> 32), w);
      if (w[0] < eps_thr) action = (uint8_t)(((uint64_t)w[1] * q->n_actions) >> 32);
      else orc_q_eval(q, x, 1, qv, &action);
    }
    if (actions_out) actions_out[k] = action;
    float r;
    orc_env_step(e, action, x, &r, NULL, NULL, two);
    if (rewards_out) rewards_out[k] = r;
    G = fmaf(disc, r, G); { volatile float d2 = disc * p->gamma; disc = d2; }
    if (recs_out) { recs_out[k] = two[0]; if (k == p->n_epochs - 1) recs_out[k + 1] = two[1]; }
  }
  if (states_out) memcpy(states_out + (size_t)p->n_epochs * ORC_STATE_DIM, x, sizeof(x));
  if (totals_out) orc_env_totals(e, totals_out);
  if (return_out) *return_out = G;
  if (util_out) orc_env_util_hist(e, util_out);
  if (n_trace_out) *n_trace_out = e->n_trace;
  orc_env_destroy(e);
  return 0;
}

/* ---------------------------------------------------------------------------------------------- ET */
double orc_et_reduce(const double *x, const double *y, const uint32_t *group, uint32_t n, uint32_t n_groups, double *et_out)
{
  double s = 0.0, t = 0.0;                       /* global means of energy and of average tardiness */
  for (uint32_t i = 0; i < n; ++i) { s += x[i]; t += y[i]; }
  s /= (double)n; t /= (double)n;
  double a = t / (2.0 * s);                      /* "we set a to be t / 2s" (L143) */
  for (uint32_t g = 0; g < n_groups; ++g) {
    double acc = 0.0; uint32_t cnt = 0;
    for (uint32_t i = 0; i < n; ++i) if (group[i] == g) { acc += (a * x[i] + y[i]) / (a + 1.0); ++cnt; }
    et_out[g] = cnt ? acc / (double)cnt : 0.0;
  }
  return a;
}
