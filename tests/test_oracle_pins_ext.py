"""Pins for the round-2 extensions of the oracle (readings #29-#32), written and checked
before any CUDA code for them:

  N  the MIG-disabled GPU as a configuration            O  the whole-GPU repartition penalty (L214)
  P  time per utilisation level (L246, Fig. 6)                          Q  the discounted return (L214)
  R  the binned 2+2m state (L210)                                       S  the BINNED policy, hourly and event-driven (L210-212)
  T  the ET metric with the global a = t / 2s (L135-143)

Expected values: tests/golden/handworked_ext.json, computed by hand (arithmetic beside each).  Mutations of
oracle/mig_oracle.c that these tests were checked to kill are listed per test.
"""
import dataclasses
from fractions import Fraction

import numpy as np
import pytest

import trace_check
from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
from util import EV_NAMES, LINEAR, SUB05, completions, events_at, golden, tiny_params

G = golden("handworked_ext.json")
G1 = golden("handworked.json")
G2 = golden("handworked_r2.json")


def as_int_keys(d):
    return {int(k): int(v) for k, v in d.items()}


# ------------------------------------------------------------------------------------------------ N: MIG disabled
def _nomig_params(**kw):
    g = G["N"]
    cfgs = tuple(tuple((s, p) for s, p in row) for row in g["configs"])
    sp = tiny_params(speeds=(LINEAR, SUB05), configs=cfgs, **kw)
    return dataclasses.replace(sp, speed_nomig=np.array(g["speed_nomig"], dtype=np.uint32), p_idle_nomig_mw=g["p_idle_nomig_mw"],
                               p_busy_nomig_mw=g["p_busy_nomig_mw"])


def test_N_mig_disabled_gpu_has_its_own_speed_and_power():
    # mutations that fail here: speed_of(8) = the 7g column (J0 completes at 150); power of size 8 from the 7g entries;
    # U += 8 instead of 7 busy units (busy_unit_s 1160, util[7] empty)
    g = G["N"]
    sp = _nomig_params()
    jobs = O.make_jobs(g["jobs"])
    r = O.rollout(sp, 0, 0, algo=g["algo"], cfg0=0, jobs=jobs, trace_cap=64, want_states=True)
    assert completions(r.trace) == as_int_keys(g["completion_nomig"])
    assert int(r.totals["tardiness_s"]) == g["tardiness"]
    assert {int(e["aux"]) for e in r.trace if e["type"] == O.EV_START} == {g["start_aux"]}
    assert int(r.recs[0]["energy_mj"]) == g["epoch0_energy_mj"] and int(r.totals["energy_mj"]) == g["day_energy_mj"]
    assert int(r.totals["busy_unit_s"]) == g["busy_unit_s"]
    assert r.util.tolist() == g["util"]
    x = r.states[1]
    assert x[23] == np.float32(g["state_3600_size_entry"]) and not x[16:23].any() and not x[24:30].any()
    # the same jobs on the MIG-enabled 7g slice: 6 % slower for the linear job only
    r7 = O.rollout(sp, 0, 0, algo=g["algo"], cfg0=1, jobs=jobs, trace_cap=64)
    assert completions(r7.trace) == as_int_keys(g["completion_7g"])
    assert int(r7.recs[0]["energy_mj"]) == 60000 * 3600 + 188243 * 150


def test_N_switching_mig_on_is_a_repartition_of_the_whole_gpu():
    # 8@0 and 7@0 are different slices: enabling MIG destroys the one and creates the other (down for the 4 s of L214)
    g = G["N"]
    sp = _nomig_params(repart_downtime_s=4)
    env = O.Env(sp, 0, 0, jobs=O.make_jobs([(3590, 0, 100, 99999)]), trace_cap=64)
    env.reset(algo=0, cfg0=0)
    env.step(0)
    env.step(1)
    tr = env.trace()
    assert events_at(tr, 3600) == [("PREEMPT", 0, 0), ("REPART", 0xFFFFFFFF, 255)]
    assert events_at(tr, 3604) == [("SLICE_UP", 0xFFFFFFFF, 0), ("START", 0, 0)]
    # 10 s at 890/s, then the rest at 840/s from 3604: rem = 84000 - 8900 = 75100 -> ceil(75100/840) = 90
    assert completions(tr) == {0: 3694}


# ------------------------------------------------------------------------------------------------ O: whole GPU down
def _run_O(all_down, algo=0):
    d = G1["D"]
    sp = dataclasses.replace(tiny_params(repart_downtime_s=d["downtime_s"], repart_energy_mj=d["repart_energy_mj"]), repart_all_down=all_down)
    jobs = O.make_jobs(d["jobs"])
    table = np.full((24, 4), d["action_epoch1"], dtype=np.uint8)
    table[0, :] = d["cfg0"]
    r = O.rollout(sp, 0, 0, algo=algo, cfg0=d["cfg0"], policy=W.POLICY_TABLE, table=table, jobs=jobs, trace_cap=256)
    return sp, jobs, r


def test_O_whole_gpu_down_requeues_every_running_job():
    # mutations that fail here: only the destroyed slices' jobs requeued (no PREEMPT of J1); unchanged slice 4g@0 stays up
    # (J1 would complete at 3675 as in D); the flag ignored in the second loop (no SLICE_UP of slot 0)
    g = G["O"]
    sp, jobs, r = _run_O(1)
    tr = r.trace
    trace_check.check_against_records(sp, G1["D"]["cfg0"], tr, r.recs, r.totals, jobs_in=jobs)
    assert completions(tr) == as_int_keys(g["completion"])
    for t in (3600, 3660, 3735):
        assert events_at(tr, t) == [tuple(e) for e in g["events_%d" % t]], t
    assert int(r.recs[0]["energy_mj"]) == g["epoch0_energy_mj"] and int(r.recs[1]["energy_mj"]) == g["epoch1_energy_mj"]
    assert int(r.recs[1]["n_preempt"]) == g["epoch1_n_preempt"]
    # flag off = hand-worked D
    _, _, r0 = _run_O(0)
    assert completions(r0.trace) == as_int_keys(G1["D"]["completion"]) and int(r0.recs[1]["energy_mj"]) == G1["D"]["epoch1_energy_mj"]


# ------------------------------------------------------------------------------------------------ P: utilisation levels
def test_P_time_per_utilisation_level():
    # mutations that fail here: util indexed by busy SLICES (D: level 2 instead of 6/7); dt added after U changed;
    # the level not integrated while every slice is down
    g = G["P"]
    _, _, rD = _run_O(0)
    assert rD.util.tolist() == g["util_D"]
    _, _, rO = _run_O(1)
    assert rO.util.tolist() == g["util_O"] and int(rO.totals["busy_unit_s"]) == g["busy_unit_s_O"]
    for r in (rD, rO):
        assert int(r.util.sum()) == int(r.totals["t_end"]) == 86400
        assert int((np.arange(8) * r.util).sum()) == int(r.totals["busy_unit_s"])


@pytest.mark.parametrize("algo", [0, 1, 2, 3, 4])
def test_P_utilisation_levels_on_generated_days(algo):
    # on any day: the levels add up to the simulated time, their first moment is the busy-unit integral, and only
    # levels that the configuration can produce are visited (cfg 3 {4g,2g,1g}: every subset sum 0..7)
    sp = W.make_params([LINEAR, SUB05], [W.dur_uniform(20, 400)] * 2, [1, 1], jobs_per_day=600, amplitude=0.6, cap=64)
    for cfg, levels in ((2, {0, 1, 2, 3, 4, 5, 6, 7}), (1, {0, 3, 4, 7}), (4, {0, 3, 6}), (0, {0, 7})):
        r = O.rollout(sp, 5, 3, algo=algo, cfg0=cfg)
        assert int(r.util.sum()) == int(r.totals["t_end"])
        assert int((np.arange(8) * r.util).sum()) == int(r.totals["busy_unit_s"])
        assert set(np.nonzero(r.util)[0].tolist()) <= levels and r.util[0] > 0


# ------------------------------------------------------------------------------------------------ Q: discounted return
def test_Q_discounted_return_by_hand():
    # mutations that fail here: gamma applied before the first reward (-17.875); G += r (gamma ignored: -50);
    # the drain's tardiness left out of the last reward
    g = G["Q"]
    sp = dataclasses.replace(tiny_params(day_s=g["n_epochs"] * 3600, n_epochs=g["n_epochs"], w_energy=g["w_energy"], w_tardy=g["w_tardy"]), gamma=g["gamma"])
    r = O.rollout(sp, 0, 0, algo=0, cfg0=0, jobs=O.make_jobs(g["jobs"]))
    assert r.rewards.tolist() == g["rewards"]
    assert r.ret == g["return"]


def test_Q_discounted_return_limits_and_bound():
    sp = W.make_params([LINEAR, SUB05], [W.dur_uniform(20, 400)] * 2, [1, 1], jobs_per_day=600, amplitude=0.6, cap=64)
    r1 = O.rollout(dataclasses.replace(sp, gamma=1.0), 5, 3, algo=1, cfg0=2)
    r0 = O.rollout(dataclasses.replace(sp, gamma=0.0), 5, 3, algo=1, cfg0=2)
    rg = O.rollout(dataclasses.replace(sp, gamma=0.9), 5, 3, algo=1, cfg0=2)
    assert r0.ret == float(r0.rewards[0])                                       # gamma = 0: the first reward, exactly
    assert np.array_equal(r1.rewards, rg.rewards)                               # the discount does not touch the rewards
    exact1 = sum(Fraction(float(x)) for x in r1.rewards)
    assert abs(Fraction(r1.ret) - exact1) <= Fraction(24, 2 ** 24) * abs(exact1)
    gam = Fraction(float(np.float32(0.9)))
    exact = sum(Fraction(float(x)) * gam ** k for k, x in enumerate(rg.rewards))
    assert abs(Fraction(rg.ret) - exact) <= Fraction(48, 2 ** 24) * sum(abs(Fraction(float(x))) * gam ** k for k, x in enumerate(rg.rewards))


# ------------------------------------------------------------------------------------------------ R: binned state
def _binned(sp, g=None):
    g = g or G["R"]
    return dataclasses.replace(sp, n_tbins=g["n_tbins"], dbin_edges=np.array(g["dbin_edges"], dtype=np.int32),
                               abin_edges=np.array(g["abin_edges"], dtype=np.int32))


def test_R_binned_state_index_by_hand():
    # mutations that fail here: v > edge instead of v >= edge; bins of the CLAMPED mean (J0: abin 2 either way, so also
    # a direct check below); first-3 in id order; code without the +1 (absent job = bin 0); time bin by epoch of the
    # NEXT hour; cfg as the innermost digit
    g, k = G["R"], G2["K"]
    sp = _binned(tiny_params(speeds=(LINEAR, SUB05), cap=k["cap"], repart_downtime_s=k["downtime_s"], repart_energy_mj=k["repart_energy_mj"]))
    env = O.Env(sp, 0, 0, jobs=O.make_jobs(k["jobs"]))
    env.reset(algo=k["algo"], cfg0=k["cfg0"])
    assert env.binned_index() == g["index_0"]
    env.step(k["actions"][0])
    assert env.binned_index() == g["index_3600"]
    env.step(k["actions"][1])
    assert env.binned_index() == g["index_7200"]


def test_R_bin_borders():
    # a job whose feature sits exactly on an edge belongs to the upper bin; one below to the lower
    sp = _binned(tiny_params())
    # durations: work = dur7*840 on the 7g slice -> mean remaining duration = dur7 at arrival
    for dur7, want_a in ((7999, 0), (8000, 1), (19999, 1), (20000, 2)):
        env = O.Env(sp, 0, 0, jobs=O.make_jobs([(3600, 0, dur7, 3600 + 5000)]))
        env.reset(algo=0, cfg0=0)
        env.step(0)          # ends at t = 3600 with the arrival processed (events at t_end belong to the step)
        assert env.n_sys() == 1
        code = 1 + 2 * 3 + want_a                              # due - t = 5000 -> dbin 2
        assert env.binned_index() == ((0 * 24 + 1) * 10 + code) * 100, (dur7, env.binned_index())
    for slack, want_d in ((-1, 0), (0, 1), (3599, 1), (3600, 2)):
        env = O.Env(sp, 0, 0, jobs=O.make_jobs([(3600, 0, 9000, 3600 + slack)]))
        env.reset(algo=0, cfg0=0)
        env.step(0)
        code = 1 + want_d * 3 + 1                              # mean duration 9000 -> abin 1
        assert env.binned_index() == ((0 * 24 + 1) * 10 + code) * 100, (slack, env.binned_index())


# ------------------------------------------------------------------------------------------------ S: BINNED policy
def _stay_table(sp):
    B = sp.binned_codes
    t = np.zeros((sp.n_configs, sp.n_tbins, B, B, B), dtype=np.uint8)
    for c in range(sp.n_configs):
        t[c] = c
    return t


def test_S_binned_policy_event_driven_reproduces_handworked_J():
    # hand-worked J (handworked.json): "empty system -> cfg 2 (id 1), otherwise cfg 3 (id 2)", decided at every arrival
    # and completion.  The same rule as a table over the binned state: first-job code 0 (no job) -> 1, any other -> 2.
    j = G1["J"]
    sp = _binned(dataclasses.replace(tiny_params(repart_downtime_s=j["downtime_s"], repart_energy_mj=j["repart_energy_mj"]), decide_on_events=1))
    t = _stay_table(sp)
    t[:, :, 0] = j["table"]["bucket0"]
    t[:, :, 1:] = j["table"]["bucket1_3"]
    jobs = O.make_jobs(j["jobs"])
    r = O.rollout(sp, 0, 0, algo=j["algo"], cfg0=j["cfg0"], policy=W.POLICY_BINNED, table=t, jobs=jobs, trace_cap=64)
    trace_check.check_against_records(sp, j["cfg0"], r.trace, r.recs, r.totals, jobs_in=jobs)
    assert [[int(e["t"]), EV_NAMES[int(e["type"])], int(e["job"]), int(e["slot"])] for e in r.trace] == j["events"]
    assert [int(e["aux"]) for e in r.trace if e["type"] == 8] == j["repart_aux"]
    assert int(r.recs[0]["energy_mj"]) == j["epoch0_energy_mj"]
    # hourly decisions only: the system is empty at every epoch start, the policy says cfg 1 = stay
    r2 = O.rollout(dataclasses.replace(sp, decide_on_events=0), 0, 0, algo=j["algo"], cfg0=j["cfg0"], policy=W.POLICY_BINNED, table=t, jobs=jobs, trace_cap=64)
    assert int(r2.totals["n_repart"]) == 0


def test_S_binned_policy_reads_the_bins_of_the_first_job():
    # the deadline bin of the first job decides: a job with more than an hour of slack leaves the configuration alone,
    # an urgent one (due within the hour) calls for the single fast slice (cfg 1 = id 0) at its arrival
    sp = _binned(dataclasses.replace(tiny_params(repart_downtime_s=4), decide_on_events=1))
    t = _stay_table(sp)
    urgent = [1 + 1 * 3 + a for a in range(3)]                 # dbin 1, any duration bin
    t[2][:, urgent] = 0
    r = O.rollout(sp, 0, 0, algo=1, cfg0=2, policy=W.POLICY_BINNED, table=t, jobs=O.make_jobs([(100, 0, 50, 9000), (5000, 0, 50, 5600)]), trace_cap=64)
    reps = [(int(e["t"]), int(e["aux"])) for e in r.trace if e["type"] == 8]
    assert reps == [(5000, (2 << 8) | 0)]
    assert [int(x) for x in r.recs["cfg"][:3]] == [2, 0, 0]


def test_S_binned_table_that_ignores_the_jobs_equals_the_tabulated_policy():
    # metamorphic pin through an independent path: a BINNED table that depends on the hour only gives the day of the
    # TABLE policy with the same hourly row (generated arrivals, every algorithm)
    sp = _binned(W.make_params([LINEAR, SUB05], [W.dur_uniform(20, 400)] * 2, [1, 1], jobs_per_day=600, amplitude=0.6, cap=64,
                               repart_downtime_s=60, repart_energy_mj=6_000_000))
    rng = np.random.default_rng(7)
    hourly = rng.integers(0, sp.n_configs, size=24).astype(np.uint8)
    tb = np.zeros((sp.n_configs, sp.n_tbins) + (sp.binned_codes,) * 3, dtype=np.uint8)
    for h in range(24):
        tb[:, h] = hourly[h]
    tt = np.repeat(hourly[:, None], 4, axis=1)
    for algo in range(5):
        a = O.rollout(sp, 9, 1, algo=algo, cfg0=3, policy=W.POLICY_BINNED, table=tb)
        b = O.rollout(sp, 9, 1, algo=algo, cfg0=3, policy=W.POLICY_TABLE, table=tt)
        assert a.totals.tobytes() == b.totals.tobytes() and a.recs.tobytes() == b.recs.tobytes()


# ------------------------------------------------------------------------------------------------ T: ET
def test_T_et_metric_by_hand():
    # mutations that fail here: a = t / s; a from per-group means; (a x + y) / a; mean over all n instead of the group
    g = G["T"]
    et, a = O.et_reduce(g["x"], g["y"], g["group"], 2)
    assert abs(a - g["a"]) < 1e-15
    for k in range(2):
        assert abs(et[k] - g["et_num"][k] / g["et_den"]) < 1e-12
    # one group: ET is linear in (x, y) with the same a
    et1, a1 = O.et_reduce(g["x"], g["y"], [0, 0, 0, 0], 1)
    assert abs(a1 - a) < 1e-15 and abs(et1[0] - (a * 25 + 3) / (a + 1)) < 1e-12
