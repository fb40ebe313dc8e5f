/*
 * migsim.h -- C ABI of libmigsim.so: the batched MIG-day simulator for NVIDIA B200 (sm_100a).
 *
 * What it computes: thousands of independent environments, each one MIG-partitioned GPU simulated over one day
 * (Lipe et al., "Energy Efficient Scheduling of AI/ML Workloads on Multi Instance GPUs with Dynamic
 * Repartitioning", CCGrid 2025 -- "PAPER.md" below is the extracted text of that paper; Lnn are its lines):
 *   problem statement, three sub-problems (partition, job priority, slice choice)
 *   MIG configurations, slice sizes 1/2/3/4/7 over 7 slots                                PAPER.md:L71-90 (Fig. 1)
 *   job model dur_js, elasticity families
 *   tardiness l_j = max(c_j - d_j, 0)
 *   ET metric (energy / tardiness scalarisation)
 *   power as a function of active compute units
 *   preemption points: every arrival and completion, all jobs re-evaluated
 *   EDF-FS, EDF-SS, LLF, LALF
 *   DQN: state, 12 actions (= target configuration), reward, repartition penalty
 *   workload: non-homogeneous Poisson arrivals, day-time peak
 * The exact readings of everything the paper leaves open are in DESIGN.md section 3.
 *
 * Conventions
 *   - plain C; every call returns 0 (MIG_OK) or a negative error code; never throws, never exits;
 *     mig_last_error() returns a thread-local message for the last failing call.
 *   - "host" pointers are read during the call and copied (the caller keeps ownership and may free them);
 *     "dev" pointers are device memory OWNED BY THE CALLER (e.g. torch tensors), valid on the handle's device; the
 *     library never allocates outputs.  NULL is allowed where stated.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls taking a stream are asynchronous on
 *     it; create / destroy / debug_set_jobs / the *_host call synchronise.
 *   - a handle is not thread-safe; there is no global state and NO CPU FALLBACK: without a CUDA device every
 *     compute call fails with MIG_ECUDA.
 *   - all simulated quantities are integers: seconds (int32), milliwatts (int32), millijoules and tardiness (int64).
 *     The only floating point is the fp32 state vector, the reward and the Q-network.
 */
#ifndef MIGSIM_H_
#define MIGSIM_H_
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MIG_OK 0
#define MIG_EINVAL (-1) /* invalid argument / parameter table */
#define MIG_ENOMEM (-2) /* host or device allocation failed */
#define MIG_ECUDA (-3)  /* CUDA runtime error (message has the CUDA string) */
#define MIG_ESTATE (-4) /* call not allowed in the handle's current state (e.g. a 25th step without reset) */

#define MIG_SLOTS 7
#define MIG_STATE_DIM 64
#define MIG_MAX_CLASSES 16
#define MIG_MAX_CONFIGS 16
#define MIG_THR_BINS 1440
#define MIG_MAX_JOBS (1u << 20) /* job ids are < 2^20 per env-day: generation stops after this many accepted jobs */

/* scheduling algorithm per environment */
enum { MIG_ALGO_EDF_FS = 0, MIG_ALGO_EDF_SS = 1, MIG_ALGO_LLF = 2, MIG_ALGO_LALF = 3,
       /* EDF-SS with restricted preemption (the variant the paper's repartitioning runs on): running jobs
        * keep their slices; waiting jobs in (due, id) order take the slowest free slice on which they finish on time, else
        * evict a job with a later (due, id) from the slowest occupied slice on which they would, else take the fastest
        * free slice, else wait (reading #26) */
       MIG_ALGO_EDF_SS_R = 4 };
/* repartitioning policy of mig_sim_rollout */
enum { MIG_POLICY_STATIC = 0, MIG_POLICY_TABLE = 1, MIG_POLICY_DQN = 2,
       /* a table over the paper's binned state ("2+2m different features: the current MIG configuration,
        * time, and the deadlines and average duration of the first m jobs ... binned", m = 3), shared by all environments;
        * DESIGN.md reading #31 */
       MIG_POLICY_BINNED = 3 };
/* slice size code of the whole GPU with MIG DISABLED (the paper's first benchmark; "6% performance
 * improvement for linear jobs ... compared to a 7g.40gb slice"): allowed at slot 0 as a configuration's only slice when
 * speed_nomig is given; 7 compute units, its own speed column and power entries (reading #29) */
#define MIG_SIZE_NOMIG 8
/* per-environment status bits */
#define MIG_ST_TRUNCATED 1u  /* t_limit_s reached with jobs still in the system */
#define MIG_ST_BAD_ACTION 2u /* an action >= n_configs was treated as "stay" */
#define MIG_ST_BAD_ALGO 4u   /* an algorithm id > MIG_ALGO_EDF_SS_R was given at reset: the env runs EDF-FS (reading #28) */
/* event types of the trace */
enum { MIG_EV_ARRIVE = 1, MIG_EV_DROP = 2, MIG_EV_START = 3, MIG_EV_PREEMPT = 4, MIG_EV_COMPLETE = 5, MIG_EV_CRIT = 6,
       MIG_EV_SLICE_UP = 7, MIG_EV_REPART = 8 };

/* Parameters of mig_sim_create: all pointers are HOST arrays, copied.  Slice-size index: 0..4 = 1g,2g,3g,4g,7g. */
typedef struct {
  uint32_t n_classes;           /* 1..16 job classes (PAPER.md:L98-102 elasticity families x duration mixes) */
  uint32_t n_configs;           /* 1..16 MIG configurations (paper: the 12 of Fig. 1) */
  const uint32_t *speed;        /* [n_classes][5] work units per second on 1g,2g,3g,4g,7g; >= 1.  dur_js = ceil(rem/speed) */
  const int32_t *dur7_q;        /* [n_classes][65] quantile table of the duration on 7g in seconds; non-decreasing, >= 1 */
  const uint32_t *class_cum;    /* [n_classes] cumulative class thresholds, non-decreasing; last = 0xFFFFFFFF */
  const uint16_t *slack_q10;    /* [n_classes][2] lo,hi of the due-date slack multiplier in Q10 (lo <= hi) */
  const uint8_t *size_at_slot;  /* [n_configs][7] size of the slice STARTING at slot p (1,2,3,4,7) or 0 */
  const uint32_t *accept_thr;   /* [1440] per-minute thinning threshold lambda(t)/lambda_max * 2^32 (PAPER.md:L222 NHPP) */
  int32_t curve_mw[8];          /* power vs number of busy compute units 0..7; may be all 0 */
  int32_t p_idle_mw[5];         /* per-slice idle power by size index (BASELINE model); may be 0 */
  int32_t p_busy_mw[5];         /* per-slice busy power by size index */
  uint64_t gap_scale_q16;       /* round(2^16 ln2 / lambda_max): exponential gap = -log2(u) * this, in Q16 seconds */
  int32_t day_s;                /* arrivals stop here (86400) */
  int32_t epoch_s;              /* decision epoch length (3600) */
  int32_t n_epochs;             /* epochs per day (24); day_s <= n_epochs * epoch_s */
  int32_t t_limit_s;            /* hard horizon of the drain after the last epoch (> n_epochs * epoch_s) */
  uint32_t cap;                 /* max jobs in system (waiting + running): 1..1024; arrivals beyond are dropped */
  uint32_t job_limit;           /* 0 = none; else generation stops after this many accepted jobs */
  int32_t repart_downtime_s;    /* new slices are down this long after a repartition (paper: 4 s, L214) */
  int64_t repart_energy_mj;     /* fixed energy per repartition */
  int32_t crit_laxity_s;        /* LLF/LALF critical-laxity threshold theta */
  uint32_t crit_max;            /* max critical-laxity preemptions per job (paper: 3), <= 15 */
  float w_energy, w_tardy;      /* reward weights: r = -(w_energy * dE + w_tardy * dT) */
  uint32_t env_base;            /* global id of local env 0 (multi-GPU sharding: Philox is keyed by global env id) */
  uint32_t decide_on_events;    /* 0: the policy decides at epoch starts only.  1: with the TABLE policy of mig_sim_rollout /
                                 * mig_sim_debug_trace the table is looked up again (row of the current epoch, load bucket of that
                                 * moment) after every tick of the day in which a job arrived or completed; a different
                                 * configuration is a repartition at that tick ("re-partitioning can happen when a
                                 * job arrives or is completed"; reading #27).  Ignored by mig_sim_step. */
  /* ---- extensions; all 0 / NULL = off.  Implemented by both kernel families (mig_sim_set_tile). */
  const uint32_t *speed_nomig;  /* [n_classes] work units per second on the whole GPU with MIG disabled (size code 8), or NULL */
  int32_t p_idle_nomig_mw;      /* idle / busy power of the MIG-disabled GPU */
  int32_t p_busy_nomig_mw;
  uint32_t repart_all_down;     /* 1: a repartition takes the WHOLE GPU down for repart_downtime_s: every running job is requeued,
                                 * every slice of the new configuration comes up at t + downtime (reading #30) */
  float gamma;                  /* discount of the return G = sum_k gamma^k r_k over the decision epochs ("discounted
                                 * rewards over time"): fp32, G = fmaf(d, r_k, G); d = d * gamma; read back by mig_sim_aux */
  uint32_t n_tbins;             /* BINNED policy: time-of-day bins, bin = min(t, day_s - 1) * n_tbins / day_s; 1..255 */
  uint32_t n_dbins, n_abins;    /* BINNED policy: deadline bins and average-duration bins, 1..8 each */
  const int32_t *dbin_edges;    /* [n_dbins - 1] ascending; the deadline feature due - t is in the first bin i with value < edge[i] */
  const int32_t *abin_edges;    /* [n_abins - 1] ascending; same rule for the mean remaining duration over the configuration's slices */
  uint32_t util_hist;           /* 1: keep the seconds spent at each utilisation level (Fig. 6); mig_sim_aux */
} mig_params_t;

/* One record per env per epoch (index n_epochs = the drain).  64 bytes. */
typedef struct {
  int64_t energy_mj;      /* energy integrated over the record's span, incl. the repartition energy */
  int64_t tardiness_s;    /* sum of max(c_j - d_j, 0) over jobs completed in the span */
  uint64_t trace_hash;    /* FNV-1a-64 of every event emitted so far (running value) */
  int32_t busy_unit_s;    /* sum over time of busy compute units (utilisation) */
  int32_t t_end;          /* simulation time at the end of the span */
  uint32_t n_events;      /* trace events emitted in the span */
  uint16_t n_arrived, n_completed, n_dropped, n_tardy, n_preempt, n_start, n_crit, n_sys_end;
  uint8_t cfg;            /* configuration in force during the span (= the action taken) */
  uint8_t repartitioned;  /* 1 if the epoch began with a repartition */
  uint8_t status;         /* MIG_ST_* so far */
  uint8_t n_running_end;
  uint32_t n_sys_max;     /* max jobs in system during the span */
  uint32_t pad_;
} mig_epoch_rec_t;

/* Per-env totals over the day + drain.  80 bytes. */
typedef struct {
  int64_t energy_mj, tardiness_s;
  uint64_t trace_hash;
  int64_t busy_unit_s;
  uint32_t n_jobs, n_completed, n_dropped, n_tardy, n_preempt, n_start, n_crit, n_events, n_repart, n_sys_max;
  int32_t t_end;
  uint32_t status;
} mig_totals_t;

/* One trace event, 16 bytes.  slot = 0xFF when not applicable; job = 0xFFFFFFFF when none. */
typedef struct { int32_t t; uint8_t type; uint8_t slot; uint16_t aux; uint32_t job; int32_t value; } mig_event_t;

/* A scripted arrival (tests): arrival tick, class, duration on 7g in seconds, absolute due date. */
typedef struct { int32_t arr; uint32_t cls; int32_t dur7; int32_t due; } mig_job_t;

typedef struct mig_sim mig_sim_t;
typedef struct mig_qnet mig_qnet_t;

const char *mig_last_error(void);
/* library / build identification, e.g. "migsim sm_100a <date>" */
const char *mig_version(void);

/* Creates a simulator of n_envs environments on the current CUDA device.  Validates every table (sizes in
 * {0,1,2,3,4,7} or 8 = MIG disabled, slices inside 7 slots and not overlapping, speed >= 1, monotone quantiles, cap in 1..1024, all
 * derived quantities inside int32) -> MIG_EINVAL with a message.  seed is the Philox key. */
int mig_sim_create(mig_sim_t **out, const mig_params_t *p, uint32_t n_envs, uint64_t seed);
int mig_sim_destroy(mig_sim_t *s);

/* Starts a new day: episode goes into the Philox counter (fresh arrivals per episode).  algo, cfg0: dev[n_envs].
 * state_out: dev[n_envs][64] fp32 initial observation, or NULL. */
int mig_sim_reset(mig_sim_t *s, uint32_t episode, const uint8_t *algo, const uint8_t *cfg0, float *state_out, void *stream);

/* One decision epoch for every env: action = target configuration (== current: stay, no cost;
 * >= n_configs: stay + MIG_ST_BAD_ACTION).  The last epoch also runs the drain.  Outputs (each dev[n_envs] or NULL):
 * state_out [n_envs][64], reward_out, energy_mj_out / tardiness_s_out (this epoch, drain included on the last),
 * rec_out (this epoch's record), drain_rec_out (written on the last epoch only).  MIG_ESTATE after n_epochs steps. */
int mig_sim_step(mig_sim_t *s, const uint8_t *action, float *state_out, float *reward_out, int64_t *energy_mj_out,
                 int64_t *tardiness_s_out, mig_epoch_rec_t *rec_out, mig_epoch_rec_t *drain_rec_out, void *stream);

/* Runs every remaining epoch of the day with the policy evaluated on the device; equals the same number of
 * mig_sim_step calls with the same actions.
 *   STATIC: stay on the current configuration.   TABLE: table dev[n_envs][n_epochs][4] u8, action =
 *   table[env][k][bucket], bucket by jobs in system (0 | <8 | <64 | else).   DQN: q + epsilon (eps-greedy from
 *   Philox stream 2), one Q forward per epoch over the state batch (scratch owned by the handle).
 *   BINNED: table dev[n_configs][n_tbins][B][B][B] u8, B = 1 + n_dbins * n_abins, ONE table for all environments, indexed
 *   by (configuration, time bin, code of the 1st, 2nd, 3rd job in (due, id) order over all jobs in system); a job's code is
 *   0 if there is no such job, else 1 + dbin * n_abins + abin.  With decide_on_events it is looked up after every tick with
 *   an arrival or a completion as well.  Thread-per-environment kernel only.
 * recs_out: dev[n_epochs+1][n_envs] or NULL.  totals_out: dev[n_envs] or NULL. */
int mig_sim_rollout(mig_sim_t *s, int policy, const uint8_t *table, const mig_qnet_t *q, float epsilon,
                    mig_epoch_rec_t *recs_out, mig_totals_t *totals_out, void *stream);

/* Per-env totals so far: dev[n_envs]. */
int mig_sim_totals(mig_sim_t *s, mig_totals_t *totals_out, void *stream);

/* Auxiliary per-env results so far (thread-per-environment kernel; MIG_ESTATE on the warp tiles), each NULL or dev:
 *   return_out dev[n_envs] fp32: the discounted return over the epochs done (params.gamma);
 *   util_s_out dev[n_envs][8] int32: seconds spent with U = 0..7 busy compute units over the day and the drain
 *   (Fig. 6; needs params.util_hist = 1, MIG_ESTATE otherwise). */
int mig_sim_aux(mig_sim_t *s, float *return_out, int32_t *util_s_out, void *stream);

/* ET metric, HOST arrays, double: x[i] = energy and y[i] = average tardiness of simulation i,
 * group[i] < n_groups the algorithm / policy it belongs to.  a = t / (2 s) with s, t the means of x and y over ALL n
 * simulations ("global mean ... across the simulations of all the experiments"); et_out[g] = mean over group g of
 * (a x_i + y_i) / (a + 1) (0 for an empty group).  a_out may be NULL.  MIG_EINVAL if n = 0, a group id is out of range
 * or the mean energy is 0. */
int mig_et_reduce(const double *x, const double *y, const uint32_t *group, uint32_t n, uint32_t n_groups, double *et_out,
                  double *a_out);

/* End-to-end convenience with HOST buffers: copies algo/cfg0/table (host[n_envs], host[n_envs][n_epochs][4] or NULL)
 * to the device, reset(episode) + rollout, copies totals (host[n_envs]) and records (host[n_epochs+1][n_envs] or
 * NULL) back, synchronises.  DQN policy allowed (q non-NULL).  A result buffer that lies in pinned, mapped host memory
 * (cudaHostAlloc / cudaHostRegister over the whole buffer) is written by the kernels directly: its bytes cross the link
 * while the launch runs and no copy follows; ordinary host memory is filled by a copy after the launch.  Same bytes
 * either way (tested). */
int mig_sim_rollout_host(mig_sim_t *s, uint32_t episode, const uint8_t *algo, const uint8_t *cfg0, int policy,
                         const uint8_t *table, const mig_qnet_t *q, float epsilon, mig_epoch_rec_t *recs_out,
                         mig_totals_t *totals_out);

/* Q-network MLP 64 -> H -> H -> n_actions, ReLU, fp32.  Host arrays, copied; W row-major [in][out].
 * Every output is accumulated in ascending k with one fused multiply-add per term (bit-reproducible).  hidden: any
 * multiple of 32 in 32..256 (MIG_EINVAL otherwise). */
int mig_qnet_create(mig_qnet_t **out, const float *W1, const float *b1, const float *W2, const float *b2,
                    const float *W3, const float *b3, uint32_t hidden, uint32_t n_actions);
int mig_qnet_destroy(mig_qnet_t *q);
/* state dev[B][64] -> q_out dev[B][n_actions] (or NULL), argmax_out dev[B] u8 lowest index on ties (or NULL). */
int mig_q_eval(const mig_qnet_t *q, const float *state, uint32_t B, float *q_out, uint8_t *argmax_out, void *stream);

/* ---- DQN training ("Deep Q-Learning, incorporating an epsilon-greedy exploration-exploitation
 * strategy and an experience replay buffer [21]", L214 "discounted rewards"; the paper gives no loss, optimiser or
 * hyper-parameter: DESIGN.md readings #33-#36).  One handle = the online network, a frozen target network (both start as
 * the given weights), a replay ring of `replay_capacity` transitions (s[64], a, r, s'[64], done) in device memory, and the
 * buffers of one training batch.  One training step on a batch of `batch` transitions:
 *     y_b = r_b + gamma (1 - done_b) max_a' Q_target(s'_b, a');   L = 1/(2 batch) sum_b (Q(s_b, a_b) - y_b)^2;
 *     theta <- theta - lr dL/dtheta            (plain squared TD error, plain SGD; the target network is not touched)
 * All matrix products (forward of both networks, backward through the activations, weight gradients) run on the tensor
 * cores as 3 x TF32 (hi/lo split of both operands, fp32 accumulation in TMEM): fp32-accurate, NOT bit-reproducible
 * against a CPU.  This is the training path; the forward that DRIVES a simulated trace stays mig_q_eval (fixed-order FFMA).
 * Tolerance against a double-precision evaluation of the same step: 1e-4 relative (tests/test_gpu_dqn.py).
 * hidden: 128 or 256; n_actions <= 16; batch: a multiple of 128.  Host weight arrays as in mig_qnet_create, copied. */
typedef struct mig_dqn mig_dqn_t;
int mig_dqn_create(mig_dqn_t **out, const float *W1, const float *b1, const float *W2, const float *b2, const float *W3,
                   const float *b3, uint32_t hidden, uint32_t n_actions, uint32_t replay_capacity, uint32_t batch,
                   float gamma, float lr, uint64_t seed);
int mig_dqn_destroy(mig_dqn_t *d);
/* Appends n transitions (dev arrays: s, s2 [n][64] fp32, a [n] u8, r [n] fp32, done [n] u8 or NULL = all 0) to the ring:
 * transition i lands in slot (head + i) mod capacity; when the ring is full the oldest are overwritten.  Typically fed
 * straight from mig_sim_step's state_out / reward_out and the actions given to it.  Asynchronous on `stream`. */
int mig_replay_push(mig_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2, const uint8_t *done,
                    uint32_t n, void *stream);
uint32_t mig_replay_size(const mig_dqn_t *d);
/* One training step on `batch` transitions sampled uniformly with replacement from the ring: index_b = (w * size) >> 32
 * with w = word 0 of Philox4x32-10(counter (b, 3, step, 0), key = seed) ("stream 3", reading #36).  loss_out: dev[1], the
 * loss before the step, or NULL.  MIG_ESTATE if the ring is empty.  Asynchronous on `stream`. */
int mig_dqn_train_step(mig_dqn_t *d, uint32_t step, float *loss_out, void *stream);
/* The same on an explicit batch: dev arrays of exactly `batch` rows (done may be NULL). */
int mig_dqn_train_on(mig_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2, const uint8_t *done,
                     float *loss_out, void *stream);
/* target <- online (device to device, asynchronous). */
int mig_dqn_sync_target(mig_dqn_t *d, void *stream);
/* Q-values of the online (which = 0) or target (1) network through the tensor-core path: state dev[n][64], n <= batch,
 * q_out dev[n][n_actions].  Within 1e-4 relative of mig_q_eval's. */
int mig_dqn_q(mig_dqn_t *d, int which, const float *state, uint32_t n, float *q_out, void *stream);
/* The same forward with NO allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, serving
 * loops, harnesses that forbid it): no handle; the scratch it needs (split weight copies, two hidden activations, padded
 * Q rows) is a file-scope static __device__ array of the library -- 4.8 MiB on every GPU that loads libmigsim.so, held
 * until the process exits -- sized for at most MIG_Q_STATIC_MAX_ROWS rows of a network with hidden <= 256.
 *   W1 dev[64][hidden], b1 dev[hidden], W2 dev[hidden][hidden], b2 dev[hidden], W3 dev[hidden][n_actions], b3
 *   dev[n_actions] (mig_qnet_create's layout, but DEVICE pointers: read on `stream`, never copied to the host); state
 *   dev[n][64]; q_out dev[n][n_actions]; state, b1 and b2 16-byte aligned.  hidden 128 or 256, n_actions 1..16.
 * Calls no cudaMalloc / cudaFree / allocating library routine: memsets, copies and kernels on `stream`, tensor maps encoded
 * on the host.  The first call on a device also takes the array's device address (cudaGetSymbolAddress) and sets the
 * kernels' shared-memory limits: make that call outside a graph capture.  MIG_EINVAL, with a message naming the limit,
 * if n > MIG_Q_STATIC_MAX_ROWS (call it on chunks of the batch) or an argument is out of range; MIG_ECUDA otherwise.
 * EVERY call on a device shares the one array: calls that overlap on the GPU (two streams, two threads, two graphs in
 * flight) race on it -- order them on one stream or with events.  Results: those of mig_dqn_q (same kernels). */
#define MIG_Q_STATIC_MAX_ROWS 2048
int mig_q_forward_static(const float *W1, const float *b1, const float *W2, const float *b2, const float *W3, const float *b3,
                         uint32_t hidden, uint32_t n_actions, const float *state, uint32_t n, float *q_out, void *stream);
/* Copies the weights of the online (0) or target (1) network to HOST arrays shaped as in mig_qnet_create; synchronises. */
int mig_dqn_get_weights(mig_dqn_t *d, int which, float *W1, float *b1, float *W2, float *b2, float *W3, float *b3);
/* Kernel launches issued through this handle so far. */
uint64_t mig_dqn_launch_count(const mig_dqn_t *d);

/* Debug / parity: re-runs ONE env for a whole day from the last reset's (episode, algo, cfg0), recording every event.
 * policy STATIC, TABLE or BINNED (table as in rollout), or actions != NULL: dev[n_epochs] explicit action sequence.
 * buf dev[cap_events]; n_out dev[1] = number of events emitted (may exceed cap_events; only the first are stored);
 * totals_out dev[1] or NULL.  Does not touch the handle's per-env state. */
int mig_sim_debug_trace(mig_sim_t *s, uint32_t env, int policy, const uint8_t *table, const uint8_t *actions,
                        mig_event_t *buf, uint32_t cap_events, uint32_t *n_out, mig_totals_t *totals_out, void *stream);
/* Scripted arrivals (host array, non-decreasing arr) replace the generator for every env; n = 0 restores it. */
int mig_sim_debug_set_jobs(mig_sim_t *s, const mig_job_t *jobs, uint32_t n);
/* The exact-division constants the kernels use for x / v (host helper, exposed for tests): x / v == v == 1 ? x :
 * (umulhi(x, m) >> sh) for every 0 <= x < 2^31. */
int mig_debug_div_magic(uint32_t v, uint32_t *m, uint32_t *sh);
/* Lanes per environment of the rollout kernel.  1 = one THREAD per environment (running jobs in the slice table, waiting
 * jobs in a sorted two-level queue, arrivals drawn before the event loop, no cross-lane traffic; 5x faster than the
 * tiles on batches that fill a B200, on a par with them below); 8 = four environments per warp in lockstep, 16, 32 = one warp per environment (north_star's layout).
 * 0 = default: 1.  Results are identical for every value (tested); only the launch geometry
 * and the memory footprint change.  Switching between 1 and {8, 16, 32} changes the layout of the saved per-env state:
 * allowed at any time, but the next call must then be mig_sim_reset (MIG_ESTATE otherwise).  Other values: MIG_EINVAL. */
int mig_sim_set_tile(mig_sim_t *s, int lanes_per_env);
/* Thread-per-environment kernel only: environments per warp (lanes 0 .. n-1 of every warp hold one each): 1, 2, 4, 8, 16
 * or 32; 0 = default: the smallest power of two that keeps a launch one resident wave, so that a small batch is spread
 * over many warps (little divergence, latency hidden) and a full batch uses every lane.  Launch geometry only: results
 * are identical for every value (tested).  Allowed between any two calls. */
int mig_sim_set_envs_per_warp(mig_sim_t *s, uint32_t envs_per_warp);
/* Thread-per-environment kernel only: capacity (records of 8 bytes per environment, rounded up to a multiple of 4) of the
 * arrival lists.  Before every launch that simulates, a generator kernel (one warp per environment, 32 thinning candidates
 * per pass) draws the arrivals of that launch's horizon into them (the arrival process does not depend
 * on the schedule).  Default, allocated by mig_sim_create: the expected number of accepted arrivals per day + 8 sigma,
 * computed from accept_thr and gap_scale_q16 (C5: 8 784 records = 70 KB per environment); if that allocation fails,
 * create fails with MIG_ENOMEM.  0 = no lists: arrivals are drawn inside the event loop, one at a time (slower).  A list
 * that is too small for a launch is simply continued that way, so ANY capacity gives the same results (tested).
 * 0xFFFFFFFF = back to the default.  Synchronises the device and reallocates; on MIG_ENOMEM the handle is left WITHOUT
 * lists (still correct, slower) and mig_last_error() says so.  Allowed between any two calls. */
int mig_sim_set_arrival_buffer(mig_sim_t *s, uint32_t entries_per_env);
/* Capacity of the arrival lists in use (records per environment); 0 = arrivals are drawn inside the event loop. */
uint32_t mig_sim_get_arrival_buffer(const mig_sim_t *s);
/* Thread-per-environment kernel only: draw the NEXT episode's arrivals ahead ("the arrival process does not
 * depend on the schedule", so a day's arrivals can be drawn before the day before it has ended).  on != 0: after a FULL-DAY
 * launch of episode e -- mig_sim_rollout straight after mig_sim_reset under a STATIC / TABLE / BINNED policy, 32
 * environments per warp -- the warps of the event loop that finish their day early draw the arrival lists of episode e + 1
 * into a second list buffer until the launch's last day ends; the next full-day launch, if its episode IS e + 1, finds them
 * in place and its generator draws only the environments that were left.  Any other call sequence (another episode,
 * mig_sim_step, a DQN rollout) simply does not use what was drawn.  Results are identical with the setting on or off
 * (tested); it costs a second list buffer (n_envs x capacity x 8 bytes; MIG_ENOMEM if that does not fit) and is off by
 * default.  Synchronises the device.  Allowed between any two calls. */
int mig_sim_set_prefetch(mig_sim_t *s, int on);
int mig_sim_get_prefetch(const mig_sim_t *s);
int mig_sim_get_tile(const mig_sim_t *s);
/* Number of kernel launches issued through this handle so far (bench.py's gpu_launches). */
uint64_t mig_sim_launch_count(const mig_sim_t *s);
/* Name of the rollout kernel that mig_sim_rollout launches with the handle's current settings, as ncu prints it
 * (bench.py's roofline.kernel; the ncu summaries under profiles/ are keyed by it).  Static string. */
const char *mig_sim_kernel_name(const mig_sim_t *s);
/* Measurement aid: with on != 0 every kernel launch of this handle is bracketed by two CUDA events on the launching
 * stream.  mig_sim_kernel_times synchronises on them, adds up the elapsed milliseconds per kernel family since its last
 * call -- ms_out[0] arrival generator, [1] rollout kernel, [2] Q-network -- with the launch counts (host arrays of 3,
 * launches_out may be NULL), and forgets them.  Results are unaffected. */
int mig_sim_set_profiling(mig_sim_t *s, int on);
int mig_sim_kernel_times(mig_sim_t *s, float ms_out[3], uint32_t launches_out[3]);

#ifdef __cplusplus
}
#endif
#endif
