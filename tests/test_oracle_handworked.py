"""Pins the oracle's scheduler / event order / energy integration / repartition against HAND-WORKED schedules.

Expected values live in tests/golden/handworked.json (each with its citation and the arithmetic that produced
it); none of them comes from running any implementation.  A dropped term, a wrong tie rule, a transposed
FS/SS choice or a missing preemption point changes at least one of these numbers.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
import trace_check
from util import CAP3, LINEAR, SUB05, cfg_idle_mw, completions, events_at, golden, tiny_params

G = golden("handworked.json")
ALGO = {"EDF-FS": 0, "EDF-SS": 1, "LLF": 2, "LALF": 3}


def run(sp, rows, algo, cfg, **kw):
    jobs = O.make_jobs(rows)
    r = O.rollout(sp, 0, 0, algo=algo, cfg0=cfg, jobs=jobs, trace_cap=256, **kw)
    trace_check.check_against_records(sp, cfg, r.trace, r.recs, r.totals, jobs_in=jobs)
    return r


def as_int_keys(d):
    return {int(k): v for k, v in d.items()}


@pytest.mark.parametrize("algo", G["A"]["algos"])
def test_A_single_machine_all_algorithms(algo):
    g = G["A"]
    sp = tiny_params(crit_laxity_s=g["crit_laxity_s"])
    r = run(sp, g["jobs"], algo, g["cfg"])
    assert completions(r.trace) == as_int_keys(g["completion"])
    assert int(r.totals["tardiness_s"]) == g["tardiness"]
    assert int(r.totals["n_preempt"]) == g["n_preempt"]
    assert int(r.recs[0]["energy_mj"]) == g["epoch0_energy_mj"]
    for k in range(1, 24):
        assert int(r.recs[k]["energy_mj"]) == 216_000_000
    assert int(r.recs[24]["energy_mj"]) == 0           # nothing left to drain
    assert int(r.totals["energy_mj"]) == g["day_energy_mj"]


@pytest.mark.parametrize("name", ["EDF-FS", "EDF-SS"])
def test_B_fastest_vs_slowest_feasible_slice(name):
    g = G["B"]
    sp = tiny_params()
    assert cfg_idle_mw(sp, g["cfg"]) == g["idle_mw"]
    r = run(sp, g["jobs"], ALGO[name], g["cfg"])
    assert completions(r.trace) == as_int_keys(g[name]["completion"])
    assert int(r.recs[0]["energy_mj"]) == g[name]["epoch0_energy_mj"]
    assert int(r.recs[0]["energy_mj"]) - g["idle_mw"] * 3600 == g[name]["dyn_energy_mj"]
    assert int(r.totals["tardiness_s"]) == 0


def test_B_ss_saves_energy():
    # EDF-SS lower energy at similar tardiness -- here -23.7 % dynamic energy, 0 tardiness both
    g = G["B"]
    assert g["EDF-SS"]["dyn_energy_mj"] < g["EDF-FS"]["dyn_energy_mj"]


@pytest.mark.parametrize("algo", G["C"]["algos"])
def test_C_arrival_preempts_and_falls_back_to_fastest(algo):
    g = G["C"]
    sp = tiny_params()
    r = run(sp, g["jobs"], algo, g["cfg"])
    assert completions(r.trace) == as_int_keys(g["completion"])
    assert events_at(r.trace, 10) == [tuple(e) for e in g["events_at_10"]]
    assert int(r.recs[0]["energy_mj"]) - g["idle_mw"] * 3600 == g["dyn_energy_mj"]
    assert cfg_idle_mw(sp, g["cfg"]) == g["idle_mw"]


def _run_D(action1):
    g = G["D"]
    sp = tiny_params(repart_downtime_s=g["downtime_s"], repart_energy_mj=g["repart_energy_mj"])
    env = O.Env(sp, 0, 0, jobs=O.make_jobs(g["jobs"]), trace_cap=256)
    env.reset(algo=g["algo"], cfg0=g["cfg0"])
    recs = []
    for k in range(24):
        a = action1 if k == 1 else (g["cfg0"] if k == 0 else action1)
        x, rew, dE, dT, rec = env.step(a)
        recs.append(rec[0].copy())
        if k == 23:
            recs.append(rec[1].copy())
    return g, sp, env, recs


def test_D_repartition_downtime_energy_and_requeue():
    g, sp, env, recs = _run_D(G["D"]["action_epoch1"])
    tr = env.trace()
    assert completions(tr) == as_int_keys(g["completion"])
    assert int(recs[0]["energy_mj"]) == g["epoch0_energy_mj"]
    assert int(recs[1]["energy_mj"]) == g["epoch1_energy_mj"]
    assert int(recs[1]["repartitioned"]) == 1 and int(recs[1]["cfg"]) == 1 and int(recs[0]["repartitioned"]) == 0
    at3600 = events_at(tr, 3600)
    assert at3600 == [("PREEMPT", 0, 4), ("REPART", 0xFFFFFFFF, 255)]
    rep = [ev for ev in tr if ev["type"] == 8][0]
    assert int(rep["aux"]) == g["repart_aux"]
    assert events_at(tr, 3660) == [("SLICE_UP", 0xFFFFFFFF, 4), ("START", 0, 4)]
    assert events_at(tr, 3675) == [("COMPLETE", 1, 0), ("PREEMPT", 0, 4), ("START", 0, 0)]
    assert int(env.totals()["tardiness_s"]) == 0
    assert int(env.totals()["n_repart"]) == 1
    trace_check.check_against_records(sp, g["cfg0"], tr, np.array(recs), env.totals())


def test_D_stay_costs_nothing():
    # PAPER.md:L212 "remain on the current configuration": no event, no cost, J0 stays on 2g until it completes
    g, sp, env, recs = _run_D(G["D"]["cfg0"])
    tr = env.trace()
    assert not [ev for ev in tr if ev["type"] in (7, 8)]
    assert int(env.totals()["n_repart"]) == 0
    # J1: 175 s on 4g -> 3675.  J0: 2g 240/s from 3500 to 3675 (rem 168000-42000=126000), then 4g: ceil(126000/480)=263 -> 3938
    assert completions(tr) == {1: 3675, 0: 3938}
    assert int(recs[1]["energy_mj"]) == 110000 * 3600 + 75 * (90943 + 36934) + 263 * 90943


def test_E_llf_pushes_short_job_late():
    g = G["E"]
    sp = tiny_params(crit_laxity_s=g["crit_laxity_s"], crit_max=g["crit_max"])
    for algo in (2, 3):                                   # cfg 1: LLF == LALF
        r = run(sp, g["jobs"], algo, g["cfg"])
        assert completions(r.trace) == as_int_keys(g["LLF"]["completion"])
        assert int(r.totals["tardiness_s"]) == g["LLF"]["tardiness"]
        assert [int(ev["t"]) for ev in r.trace if ev["type"] == 6] == g["LLF"]["crit_ticks"]
    for algo in (0, 1):
        r = run(sp, g["jobs"], algo, g["cfg"])
        assert completions(r.trace) == as_int_keys(g["EDF"]["completion"])
        assert int(r.totals["tardiness_s"]) == g["EDF"]["tardiness"]
        assert int(r.totals["n_crit"]) == 0


@pytest.mark.parametrize("name", ["LLF", "LALF"])
def test_F_llf_differs_from_lalf(name):
    g = G["F"]
    sp = tiny_params(speeds=(LINEAR, SUB05), crit_laxity_s=g["crit_laxity_s"])
    r = run(sp, g["jobs"], ALGO[name], g["cfg"])
    assert completions(r.trace) == as_int_keys(g[name]["completion"])
    assert int(r.recs[0]["energy_mj"]) - g["idle_mw"] * 3600 == g[name]["dyn_energy_mj"]
    assert int(r.totals["n_crit"]) == 0 and int(r.totals["tardiness_s"]) == 0


def test_F_edf_fs_equals_lalf_schedule_here():
    g = G["F"]
    sp = tiny_params(speeds=(LINEAR, SUB05), crit_laxity_s=g["crit_laxity_s"])
    r = run(sp, g["jobs"], 0, g["cfg"])
    assert completions(r.trace) == as_int_keys(g["LALF"]["completion"])


@pytest.mark.parametrize("algo", [0, 1, 2, 3])
def test_G_tie_between_equally_fast_slices_takes_smaller(algo):
    g = G["G"]
    sp = tiny_params(speeds=(CAP3,))
    r = run(sp, g["jobs"], algo, g["cfg"])
    starts = [ev for ev in r.trace if ev["type"] == 3]
    assert len(starts) == 1 and int(starts[0]["slot"]) == g["start_slot"] and int(starts[0]["aux"]) == 3
    assert completions(r.trace) == {0: g["completion"]}


def test_H_restricted_preemption_evicts_only_to_save_a_deadline():
    g = G["H"]
    sp = tiny_params()
    r = run(sp, g["jobs"], g["algo"], g["cfg"])
    assert completions(r.trace) == as_int_keys(g["completion"])
    assert events_at(r.trace, 10) == [tuple(e) for e in g["events_at_10"]]
    assert events_at(r.trace, 12) == [tuple(e) for e in g["events_at_12"]]
    assert [int(e["value"]) for e in r.trace if e["t"] == 12 and e["type"] == 4] == g["preempt_values_at_12"]
    assert int(r.totals["n_preempt"]) == g["n_preempt"] and int(r.totals["tardiness_s"]) == g["tardiness_s"]
    assert int(r.totals["energy_mj"]) == g["idle_mw"] * 86400 + g["dyn_energy_mj"]
    assert cfg_idle_mw(sp, g["cfg"]) == g["idle_mw"]
    # the unrestricted algorithm swaps the two running jobs at t = 10 ("switching two jobs between
    # different slices that might not result in any energy consumption or tardiness differences")
    u = run(sp, g["jobs"], ALGO["EDF-SS"], g["cfg"])
    assert int(u.totals["n_preempt"]) == g["n_preempt_unrestricted"] and int(u.totals["tardiness_s"]) == 0


def test_I_restricted_preemption_fallback_wait_and_no_eviction_of_earlier_deadlines():
    g = G["I"]
    r = run(tiny_params(), g["jobs"], g["algo"], g["cfg"])
    assert completions(r.trace) == as_int_keys(g["completion"])
    for t in (5, 6, 11, 175):
        assert events_at(r.trace, t) == [tuple(e) for e in g["events_at_%d" % t]], t
    assert int(r.totals["n_preempt"]) == g["n_preempt"] and int(r.totals["tardiness_s"]) == g["tardiness_s"]


def _table_J(g):
    t = np.zeros((24, 4), np.uint8)
    t[:, 0] = g["table"]["bucket0"]; t[:, 1:] = g["table"]["bucket1_3"]
    return t


def test_J_event_driven_decisions_repartition_at_arrival_and_completion():
    import dataclasses
    from util import EV_NAMES
    g = G["J"]
    sp = dataclasses.replace(tiny_params(repart_downtime_s=g["downtime_s"], repart_energy_mj=g["repart_energy_mj"]), decide_on_events=1)
    jobs = O.make_jobs(g["jobs"])
    r = O.rollout(sp, 0, 0, algo=g["algo"], cfg0=g["cfg0"], policy=W.POLICY_TABLE, table=_table_J(g), jobs=jobs, trace_cap=64)
    trace_check.check_against_records(sp, g["cfg0"], r.trace, r.recs, r.totals, jobs_in=jobs)
    assert [[int(e["t"]), EV_NAMES[int(e["type"])], int(e["job"]), int(e["slot"])] for e in r.trace] == g["events"]
    assert [int(e["aux"]) for e in r.trace if e["type"] == 8] == g["repart_aux"]
    assert int(r.recs[0]["energy_mj"]) == g["epoch0_energy_mj"]
    assert int(r.totals["n_repart"]) == g["n_repart"] and int(r.recs[0]["repartitioned"]) == 1 and int(r.recs[0]["cfg"]) == g["cfg0"]
    # without the flag the table is consulted at epoch starts only: the system is empty then, nothing ever changes
    sp0 = dataclasses.replace(sp, decide_on_events=0)
    r0 = O.rollout(sp0, 0, 0, algo=g["algo"], cfg0=g["cfg0"], policy=W.POLICY_TABLE, table=_table_J(g), jobs=jobs, trace_cap=64)
    assert int(r0.totals["n_repart"]) == 0


def test_speed_tables_match_survey_values():
    assert LINEAR == [120, 240, 360, 480, 840]
    assert SUB05 == [317, 449, 550, 635, 840]
    assert CAP3 == [280, 560, 840, 840, 840]
    assert W.speed_capped(2) == [420, 840, 840, 840, 840] and W.speed_capped(4) == [210, 420, 630, 840, 840]
    _, p_idle, p_busy = W.default_power()
    assert [b - i for b, i in zip(p_busy, p_idle)] == [15000, 36934, 62568, 90943, 188243]


def test_fig1_configuration_set():
    # PAPER.md:L71-90 Fig. 1: 12 configurations over 7 slots, sizes in {1,2,3,4,7}; config 5 = {3g,3g} leaves slot 3 empty
    t = W.size_at_slot_table()
    assert t.shape == (12, 7)
    covered = []
    for c in range(12):
        used = np.zeros(7, int)
        for p in range(7):
            g = int(t[c, p])
            assert g in (0, 1, 2, 3, 4, 7)
            if g:
                assert p + g <= 7
                used[p:p + g] += 1
        assert used.max() <= 1
        covered.append(int(used.sum()))
    assert covered == [7, 7, 7, 7, 6, 7, 7, 7, 7, 7, 7, 7]
    assert sorted(int(g) for g in t[3] if g) == [1, 1, 1, 4]         # config 4 = one 4g + three 1g
    assert sorted(int(g) for g in t[6] if g) == [1, 1, 2, 3]         # BASELINE C1 {3g,2g,1g,1g}
