// sim_common.h -- structures shared by the host API (migsim.cu) and the device code (sim_device.cuh).
// Part of libmigsim.so (product path).  Nothing here is shared with oracle/.
#pragma once
#include <stdint.h>

#include "../../include/migsim.h"

// sets mig_last_error()'s message and returns `code` (defined in migsim.cu; shared by the library's translation units)
int mig_fail(int code, const char *fmt, ...);

namespace migsim {

constexpr int kSlots = MIG_SLOTS;
constexpr int kWarpsPerCta = 4;
constexpr int kHeaderWords = 64;  // saved per-env header: 256 bytes

// meta word of a job-table entry: id[0:20) | class[20:24) | crit_cnt[24:28) | slot+1 [28:31)
constexpr uint32_t kIdMask = 0xFFFFFu;

// Everything the kernels read that is a table (global memory, read-only, L1/L2 resident).
struct DevTables {
  uint4 speed[MIG_MAX_CLASSES * 5];         // {v, magic m, shift (>=32: v == 1), 0}: x / v = umulhi(x, m) >> sh
  int32_t dur7_q[MIG_MAX_CLASSES * 65];
  uint32_t class_cum[MIG_MAX_CLASSES];       // padded with 0xFFFFFFFF beyond n_classes
  uint32_t slack_lo[MIG_MAX_CLASSES], slack_span[MIG_MAX_CLASSES];  // lo, hi - lo + 1
  uint32_t cfg_pack[MIG_MAX_CONFIGS];       // 7 nibbles: size of the slice starting at slot p
  uint32_t cfg_rank[MIG_MAX_CONFIGS];       // nibble p: rank of that slice among the configuration's in (size, slot) order
  uint32_t cfg_slot_of[MIG_MAX_CONFIGS];    // nibble r: start slot of the slice of rank r
  int32_t cfg_pidle[MIG_MAX_CONFIGS];       // sum of p_idle over the configuration's slices
  uint32_t thr[MIG_THR_BINS];
  uint32_t logT[257];                        // round(2^24 log2(1 + i/256))
  int32_t curve[8], p_idle[12], p_busy[12];  // p_idle/p_busy indexed by SIZE (0..8; 8 = MIG disabled), not by size index
  // extensions (readings #29, #31)
  uint4 speed_nomig[MIG_MAX_CLASSES];        // {v, magic, shift, 0} on the whole GPU with MIG disabled (size code 8)
  int32_t dbin_edges[8], abin_edges[8];      // BINNED policy: bin edges, padded with INT32_MAX
};

// Arguments of the arrival generator (gen_kernel.cuh).
struct GenArgs {
  const DevTables *tab;
  uint32_t *hdr;                       // [n_envs][kHeaderWords]
  uint2 *arr; uint32_t arr_cap;        // [n_envs][arr_cap] records
  uint32_t n_envs, env_first;
  uint32_t k0, k1, episode, env_base;  // Philox key, counter words
  uint64_t gap_scale;
  int32_t day_s, epoch_s, n_epochs, n_steps;
  uint32_t job_limit;
  // lists drawn ahead, in the tail of the previous day's event loop (mig_sim_set_prefetch; sim_thread.cuh: tail_prefetch): an
  // environment whose flag carries `pf_tag` has its list in `arr` already and its eight generator words in pf_words
  const uint32_t *pf_flag; const uint32_t *pf_words; uint32_t pf_tag;
};

// Drawing the NEXT day's arrivals in the tail of this day's event loop (mig_sim_set_prefetch; sim_thread.cuh: tail_prefetch):
// a warp whose 32 environments have finished their day claims environments one at a time and draws their lists of episode
// g.episode into g.arr (the handle's other list buffer) until every warp of the launch has finished its day.
struct PrefetchArgs {
  GenArgs g;                   // a fresh full day: generator state zero, horizon = the whole day
  uint32_t *words;             // [n_envs][kGenWords] generator words of the drawn lists
  uint32_t *flag; uint32_t tag;   // flag[env] = tag once its list and words are written
  unsigned int *claim;         // next environment to draw
  unsigned int *finished; uint32_t n_warps;   // warps that have finished their day / warps that will
  unsigned int *busy;          // [SMs][4]: warps of this launch still inside their day, per warp scheduler (warp slot & 3)
  uint32_t pace_ns;            // a drawing warp that shares its scheduler with such a warp sleeps this long before every pass
};

// Kernel arguments (by value, constant bank).
struct SimArgs {
  const DevTables *tab;
  uint32_t *hdr;        // [n_envs][64] words
  uint4 *jobtab;        // [n_envs][cap] entries {skey, meta, rem, due}
  uint4 *tab_override;  // debug trace: overflow table for the single env (cap entries) instead of jobtab
  uint32_t *hdr_override;  // debug trace: scratch header for the single env (thread-per-env kernel keeps running totals there)
  unsigned int *counter;  // dynamic env counter (zeroed before the launch)
  uint32_t n_envs, env_first;  // envs [env_first, env_first + n_envs) of the handle
  uint32_t n_classes, n_configs;
  uint32_t k0, k1, episode, env_base;  // Philox key, counter words
  uint64_t gap_scale;
  int32_t day_s, epoch_s, n_epochs, t_limit_s;
  uint32_t cap, job_limit, smem_entries;
  uint32_t envs_per_warp;  // thread-per-env kernel: active lanes per warp (1, 2, 4, ... 32): fewer = less divergence, more warps
  uint32_t ring_cap;    // thread-per-env kernel: capacity of the global part of the waiting queue (power of two >= cap)
  int32_t downtime_s; int64_t repart_energy;
  int32_t theta; uint32_t crit_max;
  float w_energy, w_tardy;
  // what to do
  int from_init;        // 1: initialise from algo/cfg0 (reset), 0: load the saved state
  int save;             // 1: write the state back
  int n_steps;          // epochs to run in this launch
  int policy;           // MIG_POLICY_STATIC / TABLE / BINNED, or explicit actions (a.actions)
  const uint8_t *algo, *cfg0;                        // from_init
  uint32_t *algo_mask;                               // thread-per-env kernel: bit i = some environment runs algorithm i (set by the reset launch)
  const uint8_t *table;                              // [n_envs][n_epochs][4]
  int ev_decide;                                     // TABLE policy: look the table up again after every tick with an arrival or a completion
  const uint8_t *actions; uint32_t act_stride_env, act_stride_k;   // action = actions[env * se + (k - k_first) * sk]
  // extensions (readings #29-#32)
  const uint8_t *bin_table;                          // BINNED policy: [n_configs][n_tbins][B][B][B], one table for all envs
  uint32_t n_tbins, n_dbins, n_abins;
  int all_down;                                      // a repartition takes the whole GPU down
  int util_hist;                                     // keep the seconds per utilisation level in the env's header
  float gamma;                                       // discount of the return kept in the env's header
  const mig_job_t *script; uint32_t n_script;
  const uint2 *arr; uint32_t arr_cap;                // thread-per-env kernel: arrival lists [n_envs][arr_cap] of 8-byte records (gen_kernel.cuh), or NULL
  int pf_on; PrefetchArgs pf;                        // thread-per-env kernel: draw the next day's lists in the launch's tail
  // outputs (NULL = skip)
  float *state_out; float *reward_out; int64_t *energy_out; int64_t *tard_out;
  mig_epoch_rec_t *recs; int32_t rec_k0; mig_epoch_rec_t *drain_rec;   // record of epoch k -> recs[(k - rec_k0) * n_envs_total + env]
  uint32_t rec_stride;                               // n_envs_total
  mig_totals_t *totals;
  mig_event_t *trace; uint32_t trace_cap; uint32_t *trace_n;
};

}  // namespace migsim
