// gen_kernel.cuh -- the arrival generator of the thread-per-environment path as its OWN kernel (
// DESIGN.md R1-R5), launched on the same stream right before sim_thread_kernel.
//
// The arrival process does not depend on the schedule, so a launch's arrivals can all be drawn before
// it simulates -- and drawing them is embarrassingly parallel over thinning CANDIDATES, where the event loop is serial:
//   * ONE WARP PER ENVIRONMENT, 128 candidates per pass: lane l draws the four consecutive candidates k + 4 l + j (Philox
//     stream 0: gap, accept, class, slack; four independent chains per lane), the integer -log2 turns w_gap into a Q16
//     gap, the lane sums its own four, ONE warp scan (SHFL.UP; 32-bit when 128 gaps fit, else 64-bit) plus the running
//     sum gives every candidate its arrival tick -- integer addition is associative, so this IS the oracle's sequential
//     accumulation;
//   * Lewis-Shedler thinning against the per-minute threshold table; a warp scan of the per-lane counts compacts the
//     accepted candidates into a per-warp shared-memory buffer in list order;
//   * the attribute pass runs over that buffer 32 at a time with every lane busy: only accepted candidates draw Philox
//     stream 1 (duration) and look their class / duration / slack up;
//   * each accepted job becomes ONE 8-BYTE record {dur7 | class | slack, tick} appended to the environment's list; the
//     32 lanes of a pass write neighbouring records (coalesced).  The event loop recomputes work = dur7 * v7[class] and
//     due = tick + max(1, dur7 * slack >> 10) when it takes the record (two multiplies) -- half the bytes of a
//     {tick, class, work, due} record through HBM.
// A candidate is COMMITTED (the saved generator state moves past it) only if it lies inside the day and the launch's
// horizon and the list still has room; generation resumes exactly at the first uncommitted candidate, in the next
// launch's generator or -- when a list is too small for its launch -- in the event loop's own one-at-a-time generator
// (EnvT::gen_next_inline).  Any list capacity therefore gives the same day (tested).
#pragma once
#include <cuda_runtime.h>

#include "philox.cuh"
#include "sim_common.h"

namespace migsim {

constexpr int kGenWarps = 8;     // environments (= warps) per CTA of the generator

// generator state of the thread-per-environment path inside the saved per-env header (word indices; sim_thread.cuh
// owns the rest of the layout)
enum { HG_PK = 1 /* epoch in the low byte */, HG_GK = 6, HG_GT_LO, HG_GT_HI, HG_GDONE, HG_NACC,
       HG_ACOUNT = 32 /* records in this launch's list */, HG_AMORE /* the list filled up before the horizon */, HG_AID0 /* job id of record 0 */ };

constexpr int kGenWords = 8;     // generator words of an environment: HG_GK .. HG_NACC (5), HG_ACOUNT .. HG_AID0 (3)

// the tables the generator reads (shared-memory copies in gen_arrivals_kernel, the global originals in the event loop's tail)
struct GenTabs { const uint32_t *thr; const int32_t *dur7_q; const uint32_t *class_cum, *slack_lo, *slack_span, *logT; };

constexpr int kGenRun = 4;       // consecutive candidates per lane and pass: 128 per warp pass, four independent Philox chains per lane
static_assert(kGenRun <= 4, "the per-lane flag word holds three nibbles");
struct GenPend { uint32_t k, tick, wz, ww; };   // an accepted candidate waiting for its attributes: index, arrival tick, class word, slack word

struct GenSmem {
  GenPend pend[kGenWarps][32 * kGenRun];
  uint32_t thr[MIG_THR_BINS];
  int32_t dur7_q[MIG_MAX_CLASSES * 65];
  uint32_t class_cum[MIG_MAX_CLASSES];      // padded with 0xFFFFFFFF beyond n_classes
  uint32_t slack_lo[MIG_MAX_CLASSES], slack_span[MIG_MAX_CLASSES];
  uint32_t logT[257];
};

// arrival record: x = dur7[0:25) | class[25:29) | slack_q10 bits 13..15 [29:32);  y = tick[0:17) | slack_q10 bits 0..12 [17:30)
__device__ __forceinline__ uint2 pack_arrival(uint32_t tick, uint32_t cls, uint32_t dur7, uint32_t slack) {
  return make_uint2(dur7 | (cls << 25) | ((slack >> 13) << 29), tick | ((slack & 0x1FFFu) << 17));
}

// E24 = -log2((w|1) / 2^32) * 2^24 by table + linear interpolation, all integer (R3)
__device__ __forceinline__ uint32_t neglog2_q24_tab(uint32_t w, const uint32_t *logT) {
  const uint32_t m = w | 1u;
  const int lz = __clz((int)m);
  const uint32_t y = m << lz;
  const uint32_t i = (y >> 23) & 0xFFu, f = (y >> 7) & 0xFFFFu;
  const uint32_t T0 = logT[i], T1 = logT[i + 1];
  const uint32_t L = T0 + (uint32_t)(((unsigned long long)(T1 - T0) * f) >> 16);
  return ((uint32_t)(1 + lz) << 24) - L;
}

// first c with w <= cum[c] over 16 non-decreasing thresholds whose last is 0xFFFFFFFF: four dependent compares
__device__ __forceinline__ uint32_t class_of(uint32_t w, const uint32_t *cum) {
  uint32_t c = (w > cum[7]) ? 8u : 0u;
  c += (w > cum[c + 3]) ? 4u : 0u;
  c += (w > cum[c + 1]) ? 2u : 0u;
  c += (w > cum[c]) ? 1u : 0u;
  return c;
}




// One environment's arrivals from the generator state (epoch, k, done, nacc, T) up to the launch's horizon, by one warp
// (every condition in the loop is warp-uniform).  `pend(i)`: the warp's buffer of 32 * kGenRun accepted candidates; `pace()` runs
// before every pass (the event loop's tail yields to the warps that still simulate);
// o_state[5] receives {k, T lo, T hi, done, nacc}, o_list[3] {records in the list, list filled up, job id of record 0}.
template <class Pend, class Pace>
__device__ __forceinline__ void gen_env(const GenArgs &a, const GenTabs &tb, Pend pend, Pace pace, uint32_t lane, uint32_t env_g, uint2 *out,
                                        int epoch, uint32_t k, uint32_t done, uint32_t nacc, unsigned long long T,
                                        uint32_t *o_state, uint32_t *o_list) {
  const uint32_t id0 = nacc, limit = a.job_limit ? min(a.job_limit, MIG_MAX_JOBS) : MIG_MAX_JOBS;
  uint32_t count = 0, more = 0;
  if (epoch < a.n_epochs && !done) {
    const unsigned long long horizon = (unsigned long long)(min(epoch + a.n_steps, a.n_epochs) * a.epoch_s);
    // a gap is at most 32 gap_scale (E24 <= 32 << 24): with gap_scale < 2^20 the sum of a pass of 128 is < 2^32
    const bool narrow = a.gap_scale < (1ull << 20);
    for (;;) {                                                    // every condition below is warp-uniform
      if (nacc >= limit) break;
      if (count >= a.arr_cap) { more = 1; break; }
      pace();
      // ---- lane l draws the kGenRun consecutive candidates k + kGenRun l + j (Philox stream 0: gap, accept, class, slack)
      const uint32_t kb = k + lane * kGenRun;
      uint32_t wy[kGenRun], wz[kGenRun], ww[kGenRun];
      unsigned long long s[kGenRun];                              // inclusive sums of the lane's own gaps
      unsigned long long run = 0;
#pragma unroll
      for (int j = 0; j < kGenRun; ++j) {
        const uint4 w = philox4x32_10(kb + (uint32_t)j, 0u, env_g, a.episode, a.k0, a.k1);
        run += ((unsigned long long)neglog2_q24_tab(w.x, tb.logT) * a.gap_scale) >> 24;
        s[j] = run; wy[j] = w.y; wz[j] = w.z; ww[j] = w.w;
      }
      // ---- exclusive warp scan of the lane totals (integer: the same sums as the oracle's sequential accumulation)
      unsigned long long incl;
      if (narrow) {
        uint32_t g32 = (uint32_t)run;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t o = __shfl_up_sync(0xffffffffu, g32, d);
          if (lane >= (uint32_t)d) g32 += o;
        }
        incl = g32;
      } else {
        incl = run;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const unsigned long long o = __shfl_up_sync(0xffffffffu, incl, d);
          if (lane >= (uint32_t)d) incl += o;
        }
      }
      const unsigned long long base = T + (incl - run);
      // ---- thinning (Lewis-Shedler) per candidate; flags: bit j = inside the day, bit 4 + j = also inside the horizon, bit 8 + j = accepted
      uint32_t tick[kGenRun], fl = 0, n_acc_l = 0;
#pragma unroll
      for (int j = 0; j < kGenRun; ++j) {
        const unsigned long long tk = (base + s[j]) >> 16;
        const bool in_day = tk < (unsigned long long)a.day_s;     // arrivals stop at the end of the day
        const bool ok = in_day && tk <= horizon;
        tick[j] = (uint32_t)tk;
        const bool acc = ok && wy[j] <= tb.thr[(ok ? (uint32_t)tk : 0u) / 60u];
        fl |= (in_day ? 1u : 0u) << j | (ok ? 1u : 0u) << (4 + j) | (acc ? 1u : 0u) << (8 + j);
        n_acc_l += acc ? 1u : 0u;
      }
      uint32_t before = n_acc_l;                                  // accepted among the EARLIER candidates of the pass (lane-major order)
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, before, d);
        if (lane >= (uint32_t)d) before += o;
      }
      before -= n_acc_l;
      // ---- commit a prefix of the pass: inside the horizon and room left in the list (ticks and `before` are monotone)
      const uint32_t room = min(a.arr_cap - count, limit - nacc);
      uint32_t nc_l = 0, na_l = 0, b = before;
#pragma unroll
      for (int j = 0; j < kGenRun; ++j) {
        const bool commit = ((fl >> (4 + j)) & 1u) && b < room;
        const bool acc = (fl >> (8 + j)) & 1u;
        nc_l += commit ? 1u : 0u;
        if (commit && acc) {                                      // park it for the attribute pass, in list order
          pend(b) = GenPend{kb + (uint32_t)j, tick[j], wz[j], ww[j]};
          ++na_l;
        }
        b += acc ? 1u : 0u;
      }
      const uint32_t nc = __reduce_add_sync(0xffffffffu, nc_l), na = __reduce_add_sync(0xffffffffu, na_l);
      __syncwarp();
      // ---- job attributes (R5) of the accepted candidates, 32 per trip with every lane busy: class, Philox stream 1
      // (duration), slack; one coalesced 8-byte record each
      for (uint32_t i = lane; i < na; i += 32u) {
        const GenPend e = pend(i);
        const uint32_t c = class_of(e.wz, tb.class_cum);
        const uint4 wd = philox4x32_10(e.k, 1u, env_g, a.episode, a.k0, a.k1);
        const uint32_t qi = wd.x >> 26, f = (wd.x >> 16) & 0x3FFu;
        const int q0 = tb.dur7_q[c * 65 + qi], q1 = tb.dur7_q[c * 65 + qi + 1];
        const int dur7 = q0 + (int)(((long long)(q1 - q0) * (long long)f) >> 10);
        const uint32_t slack = tb.slack_lo[c] + __umulhi(e.ww, tb.slack_span[c]);
        __stcg(&out[count + i], pack_arrival(e.tick, c, (uint32_t)dur7, slack));   // streamed past L1
      }
      __syncwarp();
      count += na; nacc += na;
      if (nc) {                                                   // the generator moves past the committed candidates
        const uint32_t lc = (nc - 1u) / kGenRun, jc = (nc - 1u) % kGenRun;
        unsigned long long tl = base + s[0];
#pragma unroll
        for (int j = 1; j < kGenRun; ++j) tl = jc == (uint32_t)j ? base + s[j] : tl;
        T = __shfl_sync(0xffffffffu, tl, (int)lc); k += nc;
      }
      if (nc < 32u * kGenRun) {                                   // the first uncommitted candidate says why we stop
        const uint32_t f1 = __shfl_sync(0xffffffffu, fl, (int)(nc / kGenRun)), j1 = nc % kGenRun;
        const bool s_in_day = (f1 >> j1) & 1u, s_ok = (f1 >> (4 + j1)) & 1u;
        if (!s_in_day) done = 1;                                  // end of the day
        else if (s_ok && nacc < limit) more = 1;                  // inside the horizon: the list is full
        break;
      }
    }
  }
  if (lane == 0) {
    o_state[0] = k; o_state[1] = (uint32_t)T; o_state[2] = (uint32_t)(T >> 32); o_state[3] = done; o_state[4] = nacc;
    o_list[0] = count; o_list[1] = more; o_list[2] = id0;
  }
}

__global__ void __launch_bounds__(kGenWarps * 32, 3) gen_arrivals_kernel(const GenArgs a) {
  __shared__ GenSmem sm;
  const uint32_t lane = threadIdx.x & 31u, li = blockIdx.x * kGenWarps + (threadIdx.x >> 5);
  const uint32_t env = a.env_first + (li < a.n_envs ? li : 0u);
  uint32_t *hdr = a.hdr + (size_t)env * kHeaderWords;
  // drawn ahead (mig_sim_set_prefetch): the eight generator words move into the header, the list is in place
  const bool ahead = li < a.n_envs && a.pf_flag && a.pf_flag[env] == a.pf_tag;
  if (ahead && lane < (uint32_t)kGenWords) hdr[lane < 5u ? HG_GK + lane : HG_ACOUNT + (lane - 5u)] = a.pf_words[(size_t)env * kGenWords + lane];
  if (!__syncthreads_or(li < a.n_envs && !ahead)) return;          // nothing to draw in this CTA
  {
    const DevTables *tb = a.tab;
    for (int i = threadIdx.x; i < MIG_THR_BINS; i += kGenWarps * 32) sm.thr[i] = tb->thr[i];
    for (int i = threadIdx.x; i < MIG_MAX_CLASSES * 65; i += kGenWarps * 32) sm.dur7_q[i] = tb->dur7_q[i];
    for (int i = threadIdx.x; i < 257; i += kGenWarps * 32) sm.logT[i] = tb->logT[i];
    if (threadIdx.x < MIG_MAX_CLASSES) {
      sm.class_cum[threadIdx.x] = tb->class_cum[threadIdx.x];
      sm.slack_lo[threadIdx.x] = tb->slack_lo[threadIdx.x]; sm.slack_span[threadIdx.x] = tb->slack_span[threadIdx.x];
    }
  }
  __syncthreads();
  if (li >= a.n_envs || ahead) return;
  const GenTabs tb{sm.thr, sm.dur7_q, sm.class_cum, sm.slack_lo, sm.slack_span, sm.logT};
  GenPend *const mine = sm.pend[threadIdx.x >> 5];                // this warp's accepted candidates of the pass
  const unsigned long long T = (unsigned long long)hdr[HG_GT_LO] | ((unsigned long long)hdr[HG_GT_HI] << 32);
  gen_env(a, tb, [mine](uint32_t i) -> GenPend & { return mine[i]; }, [] {}, lane, a.env_base + env, a.arr + (size_t)env * a.arr_cap,
          (int)(hdr[HG_PK] & 0xFFu), hdr[HG_GK], hdr[HG_GDONE], hdr[HG_NACC], T, hdr + HG_GK, hdr + HG_ACOUNT);
}

}  // namespace migsim
