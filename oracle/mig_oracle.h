/*
 * mig_oracle.h -- CPU ORACLE of the batched MIG-day simulator.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded, event-by-event implementation of what the paper defines
 * (Lipe et al., "Energy Efficient Scheduling of AI/ML Workloads on Multi Instance GPUs with
 * Dynamic Repartitioning", CCGrid 2025; /root/reference/PAPER.md at authoring time) under the
 * readings listed in DESIGN.md section 3.  It shares NO code with the CUDA library
 * (paper_2606_25082_b200/csrc, include/migsim.h): own structs, own Philox, own log table.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py (hand-worked schedules,
 * invariants, brute force, closed forms, an independent Philox) EXCEPT numeric agreement with the
 * paper's Tables II/III and Figs. 3-11, whose inputs (Alibaba trace rates, A100 power curve, trained
 * weights) are not available: "parity unpinned" against those results.
 */
#ifndef MIG_ORACLE_H_
#define MIG_ORACLE_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_SLOTS 7
#define ORC_STATE_DIM 64
#define ORC_MAX_JOBS (1u << 20) /* ids are < 2^20: generation stops after this many accepted jobs */

/* status flags */
#define ORC_ST_TRUNCATED 1u  /* t_limit_s reached with jobs still in system */
#define ORC_ST_BAD_ACTION 2u /* an action >= n_configs was treated as "stay" */
#define ORC_ST_BAD_ALGO 4u   /* an algorithm id > 4 was given at reset: the env runs EDF-FS (reading #28) */

/* event types */
enum { ORC_EV_ARRIVE = 1, ORC_EV_DROP = 2, ORC_EV_START = 3, ORC_EV_PREEMPT = 4, ORC_EV_COMPLETE = 5,
       ORC_EV_CRIT = 6, ORC_EV_SLICE_UP = 7, ORC_EV_REPART = 8 };

enum { ORC_ALGO_EDF_FS = 0, ORC_ALGO_EDF_SS = 1, ORC_ALGO_LLF = 2, ORC_ALGO_LALF = 3,
       ORC_ALGO_EDF_SS_R = 4 /* EDF-SS with restricted preemption */ };
enum { ORC_POLICY_STATIC = 0, ORC_POLICY_TABLE = 1, ORC_POLICY_DQN = 2,
       ORC_POLICY_BINNED = 3 /* table over the paper's binned 2+2m state, shared by all envs */ };
#define ORC_SIZE_NOMIG 8 /* slice size code of the whole GPU with MIG disabled */

typedef struct {
  uint32_t n_classes, n_configs;
  const uint32_t *speed;        /* [n_classes][5] work units / s on 1g,2g,3g,4g,7g */
  const int32_t *dur7_q;        /* [n_classes][65] */
  const uint32_t *class_cum;    /* [n_classes] */
  const uint16_t *slack_q10;    /* [n_classes][2] */
  const uint8_t *size_at_slot;  /* [n_configs][7] */
  const uint32_t *accept_thr;   /* [1440] */
  int32_t curve_mw[8];
  int32_t p_idle_mw[5];
  int32_t p_busy_mw[5];
  uint64_t gap_scale_q16;
  int32_t day_s, epoch_s, n_epochs, t_limit_s;
  uint32_t cap, job_limit;
  int32_t repart_downtime_s;
  int64_t repart_energy_mj;
  int32_t crit_laxity_s;
  uint32_t crit_max;
  float w_energy, w_tardy;
  uint32_t decide_on_events;    /* TABLE / BINNED policy: also decide after every tick with an arrival or a completion */
  /* --- round-2 extensions; all 0 / NULL = off (readings #29-#32) ------------------------------------ */
  const uint32_t *speed_nomig;  /* [n_classes] work units / s on the whole GPU with MIG DISABLED, slice size code 8, or NULL */
  int32_t p_idle_nomig_mw, p_busy_nomig_mw;
  uint32_t repart_all_down;     /* 1: a repartition takes the WHOLE GPU down for repart_downtime_s, every running job is requeued */
  float gamma;                  /* discount of the return sum_k gamma^k r_k ("discounted rewards over time") */
  uint32_t n_tbins, n_dbins, n_abins; /* BINNED policy: time-of-day bins, deadline bins, average-duration bins */
  const int32_t *dbin_edges;    /* [n_dbins - 1] ascending: the deadline feature due - t falls in the first bin i with value < edge[i] */
  const int32_t *abin_edges;    /* [n_abins - 1] ascending, same rule for the mean remaining duration over the configuration's slices */
} orc_params_t;

typedef struct { int32_t arr; uint32_t cls; int32_t dur7; int32_t due; } orc_job_in_t;

typedef struct { int32_t t; uint8_t type; uint8_t slot; uint16_t aux; uint32_t job; int32_t value; } orc_event_t;

typedef struct {
  int64_t energy_mj, tardiness_s;
  uint64_t trace_hash;
  int32_t busy_unit_s, t_end;
  uint32_t n_events;
  uint16_t n_arrived, n_completed, n_dropped, n_tardy, n_preempt, n_start, n_crit, n_sys_end;
  uint8_t cfg, repartitioned, status, n_running_end;
  uint32_t n_sys_max;
  uint32_t pad_;
} orc_epoch_rec_t; /* 64 bytes */

typedef struct {
  int64_t energy_mj, tardiness_s;
  uint64_t trace_hash;
  int64_t busy_unit_s;
  uint32_t n_jobs, n_completed, n_dropped, n_tardy, n_preempt, n_start, n_crit, n_events, n_repart, n_sys_max;
  int32_t t_end;
  uint32_t status;
} orc_totals_t; /* 80 bytes */

typedef struct {
  uint32_t n_actions, hidden;
  const float *W1, *b1, *W2, *b2, *W3, *b3; /* [64][H] [H] [H][H] [H] [H][A] [A] */
} orc_qnet_t;

typedef struct orc_env orc_env_t;

/* --- pieces exposed so that tests can pin them one by one ------------------------------------ */
void orc_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]);
uint32_t orc_neglog2_q24(uint32_t w);                    /* E24 = -log2((w|1) / 2^32) * 2^24 (reading R3) */
void orc_log_table(uint32_t out[257]);                   /* T[i] = round(2^24 log2(1 + i/256)) */
uint64_t orc_fnv1a_words(uint64_t h, const uint32_t w[4]);

/* --- one environment ------------------------------------------------------------------------- */
orc_env_t *orc_env_create(const orc_params_t *p, uint64_t seed, uint32_t env_id);
void orc_env_destroy(orc_env_t *e);
void orc_env_set_jobs(orc_env_t *e, const orc_job_in_t *jobs, uint32_t n); /* scripted arrivals replace the generator */
void orc_env_set_trace(orc_env_t *e, orc_event_t *buf, uint32_t cap_events); /* record every event (n via orc_env_n_events) */
uint32_t orc_env_n_events(const orc_env_t *e);
void orc_env_reset(orc_env_t *e, uint32_t episode, uint8_t algo, uint8_t cfg0);
/* one epoch (plus the drain after the last one).  rec_out: 2 records (epoch, drain) or NULL. Returns 0, or -1 when the day is over. */
int orc_env_step(orc_env_t *e, uint8_t action, float *state_out, float *reward_out, int64_t *energy_out,
                 int64_t *tardiness_out, orc_epoch_rec_t *rec_out);
void orc_env_observe(const orc_env_t *e, float *state_out);
void orc_env_totals(const orc_env_t *e, orc_totals_t *out);
uint32_t orc_env_n_sys(const orc_env_t *e);

/* whole day for one env: reset + n_epochs steps with the policy evaluated inside.
 * table: [n_epochs][4] for this env (TABLE); q + epsilon (DQN).  recs_out: [n_epochs+1] or NULL.
 * states_out: [n_epochs+1][64] (state before each step, then final) or NULL; actions_out/rewards_out: [n_epochs] or NULL. */
int orc_rollout(const orc_params_t *p, uint64_t seed, uint32_t env_id, uint32_t episode, uint8_t algo, uint8_t cfg0,
                int policy, const uint8_t *table, const orc_qnet_t *q, float epsilon,
                const orc_job_in_t *jobs, uint32_t n_jobs,
                orc_epoch_rec_t *recs_out, orc_totals_t *totals_out,
                orc_event_t *trace_buf, uint32_t trace_cap, uint32_t *n_trace_out,
                float *states_out, uint8_t *actions_out, float *rewards_out);

/* orc_rollout with the round-2 outputs.  policy BINNED: table = the shared [n_configs][n_tbins][B][B][B] u8 table,
 * B = 1 + n_dbins * n_abins.  return_out: the discounted return sum_k gamma^k r_k, accumulated in fp32 as
 * G = fmaf(d, r_k, G); d = d * gamma (d starts at 1), or NULL.  util_out: [8] seconds spent with U = 0..7 busy compute
 * units over the day and the drain (Fig. 6), or NULL. */
int orc_rollout_ex(const orc_params_t *p, uint64_t seed, uint32_t env_id, uint32_t episode, uint8_t algo, uint8_t cfg0,
                   int policy, const uint8_t *table, const orc_qnet_t *q, float epsilon,
                   const orc_job_in_t *jobs, uint32_t n_jobs,
                   orc_epoch_rec_t *recs_out, orc_totals_t *totals_out,
                   orc_event_t *trace_buf, uint32_t trace_cap, uint32_t *n_trace_out,
                   float *states_out, uint8_t *actions_out, float *rewards_out,
                   float *return_out, int32_t *util_out);
/* index of the environment's present state in the BINNED policy's table (configuration, time, deadline
 * and average duration of the first m = 3 jobs, binned) */
uint32_t orc_env_binned_index(const orc_env_t *e);
void orc_env_util_hist(const orc_env_t *e, int32_t out[8]);

/* ET metric: x[i] = energy, y[i] = average tardiness of simulation i, group[i] < n_groups = the
 * algorithm it belongs to.  a = t / (2 s) with s, t the GLOBAL means of x and y over all n simulations;
 * et_out[g] = mean over the simulations of group g of (a x + y) / (a + 1).  Returns a. */
double orc_et_reduce(const double *x, const double *y, const uint32_t *group, uint32_t n, uint32_t n_groups, double *et_out);

/* Q-network forward, fp32, one fmaf per term in ascending k; argmax lowest index on ties. */
void orc_q_eval(const orc_qnet_t *q, const float *state, uint32_t B, float *q_out, uint8_t *argmax_out);
/* the same network in double precision with plain a*b+c (for the 1e-4 relative bound) */
void orc_q_eval_f64(const orc_qnet_t *q, const float *state, uint32_t B, double *q_out);

/* --- DQN training step (dqn_oracle.c; readings #33-#36), double precision ----------------- */
typedef struct orc_dqn orc_dqn_t;
size_t orc_dqn_n_params(uint32_t hidden, uint32_t n_actions);    /* flat order: W1 [64][H], b1, W2 [H][H], b2, W3 [H][A], b3 */
orc_dqn_t *orc_dqn_create(const orc_qnet_t *init, double gamma, double lr);   /* online = target = init */
void orc_dqn_destroy(orc_dqn_t *d);
void orc_dqn_sync_target(orc_dqn_t *d);                           /* target <- online */
void orc_dqn_get(const orc_dqn_t *d, int which, double *flat);    /* which: 0 online, 1 target */
void orc_dqn_set(orc_dqn_t *d, int which, const double *flat);
void orc_dqn_q(const orc_dqn_t *d, int which, const float *s, uint32_t B, double *q_out);
/* L = 1/(2B) sum_b (Q(s_b, a_b) - (r_b + gamma (1 - done_b) max_a' Q_target(s'_b, a')))^2 and dL/d(online parameters) */
double orc_dqn_loss_grad(const orc_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2,
                         const uint8_t *done, uint32_t B, double *grad);
double orc_dqn_train_step(orc_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2,
                          const uint8_t *done, uint32_t B);       /* online -= lr * grad; returns the loss before the step */
/* replay sampling: idx_b = (word 0 of Philox(counter (b, 3, step, 0), key seed) * size) >> 32 */
void orc_replay_sample(uint64_t seed, uint32_t step, uint32_t size, uint32_t B, uint32_t *idx_out);

#ifdef __cplusplus
}
#endif
#endif
