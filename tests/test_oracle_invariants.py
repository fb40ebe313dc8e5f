"""Conservation invariants, the paper's equivalence statements, brute-force optimality and closed forms.

* north_star invariants: every job finishes exactly once, slice capacities never exceeded, energy equals the sum of
  per-interval power x duration -- checked by tests/trace_check.py, an independent replay that knows no scheduling rule;
* on configurations made of one slice size (cfg 1, cfg 5) the EDF variants coincide and the LLF variants
  coincide;  PAPER.md:L77: cfg 1 behaves as a single machine;
* textbook: on a single machine EDF (Jackson's EDD / Horn's preemptive EDF) minimises the maximum lateness -- brute force
  over all orders / all unit-slot schedules of <= 5 jobs;
* closed forms for sparse arrivals.
"""
import itertools

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
import trace_check
from util import LINEAR, completions, tiny_params, trace_tuple


def _small(wl_fn, n):
    return wl_fn(n)


@pytest.mark.parametrize("name,n_env", [("C1", 1), ("C2", 48), ("C3", 12), ("C4", 6), ("C5", 2)])
def test_invariants_on_baseline_workloads(name, n_env):
    wl = W.CONFIGS[name](n_env)
    sp = wl.params
    for e in range(n_env):
        table = None if wl.table is None else wl.table[e]
        r = O.rollout(sp, wl.seed, e, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy, table=table,
                      qnet=wl.qnet, epsilon=wl.epsilon, trace_cap=400000, want_states=True)
        assert int(r.totals["status"]) == 0
        trace_check.check_against_records(sp, int(wl.cfg0[e]), r.trace, r.recs, r.totals)
        assert int(r.totals["n_jobs"]) == int(r.totals["n_completed"]) + int(r.totals["n_dropped"])
        # hash of the trace recomputed from the records
        h = 0xcbf29ce484222325
        for ev in r.trace:
            w = [int(ev["t"]) & 0xFFFFFFFF, int(ev["type"]) | (int(ev["slot"]) << 8) | (int(ev["aux"]) << 16), int(ev["job"]),
                 int(ev["value"]) & 0xFFFFFFFF]
            for x in w:
                h = ((h ^ x) * 0x100000001b3) & 0xFFFFFFFFFFFFFFFF
        assert h == int(r.totals["trace_hash"])
        # actions: static = stay; table = table[k][bucket]; record cfg follows the action
        for k in range(sp.n_epochs):
            assert int(r.recs[k]["cfg"]) == int(r.actions[k])
        if wl.policy == W.POLICY_STATIC:
            assert np.all(r.actions == wl.cfg0[e]) and int(r.totals["n_repart"]) == 0
        # state vector sanity: one-hot hour, constant 1, exact small values
        for k in range(sp.n_epochs + 1):
            x = r.states[k]
            hour = k % 24 if k < sp.n_epochs else (int(r.totals["t_end"]) // 3600) % 24      # last one: after the drain
            assert x[63] == 1.0 and x[30:54].sum() == 1.0 and x[30 + hour] == 1.0
            assert x[54] * 64 == x[:16].sum()
        # reward = -(w_E * f32(dE) + w_T * f32(dT)) with the drain added to the last epoch
        for k in range(sp.n_epochs):
            dE = int(r.recs[k]["energy_mj"]) + (int(r.recs[k + 1]["energy_mj"]) if k == sp.n_epochs - 1 else 0)
            dT = int(r.recs[k]["tardiness_s"]) + (int(r.recs[k + 1]["tardiness_s"]) if k == sp.n_epochs - 1 else 0)
            ref = -(np.float32(sp.w_energy) * np.float32(dE) + np.float32(sp.w_tardy) * np.float32(dT))
            assert np.float32(r.rewards[k]) == np.float32(ref)


def _restricted_day(e, cfg, table=None):
    wl = W.config_c3(8)
    r = O.rollout(wl.params, 11, e, algo=4, cfg0=cfg, policy=W.POLICY_STATIC if table is None else W.POLICY_TABLE, table=table,
                  trace_cap=200000)
    assert int(r.totals["status"]) == 0
    trace_check.check_against_records(wl.params, cfg, r.trace, r.recs, r.totals)
    return wl.params, r


@pytest.mark.parametrize("cfg", [1, 2, 6, 9, 11])
def test_restricted_preemption_properties(cfg):
    """PAPER.md:L198-204, reading #26, checked on the trace alone: (1) a job is never moved between slices while it
    runs; (2) outside a repartition every PREEMPT is followed at once by the START, on the same slice, of a job with
    an earlier (due, id) that completes there by its due date; (3) far fewer preemptions than unrestricted EDF-SS
    (the paper reports 63-99 % fewer, Fig. 4) at a similar tardiness."""
    sp, r = _restricted_day(3, cfg)
    tr = r.trace
    due, cls, where = {}, {}, {}
    speed = np.asarray(sp.speed).reshape(-1, 5)
    n_evict = 0
    for i, ev in enumerate(tr):
        ty, job, slot, t = int(ev["type"]), int(ev["job"]), int(ev["slot"]), int(ev["t"])
        if ty == 1:
            due[job], cls[job] = int(ev["value"]), int(ev["aux"])
        elif ty == 3:
            assert job not in where, "a running job was started again without a PREEMPT"
            where[job] = slot
        elif ty == 5:
            del where[job]
        elif ty == 4:
            assert where.pop(job) == slot
            nxt = tr[i + 1]
            assert int(nxt["type"]) == 3 and int(nxt["slot"]) == slot and int(nxt["t"]) == t
            j2 = int(nxt["job"])
            assert (due[j2], j2) < (due[job], job)
            v = int(speed[cls[j2]][W.SIZE_INDEX[int(nxt["aux"])]])
            assert t + -(-int(nxt["value"]) // v) <= due[j2], "the evicting job does not make its deadline there"
            n_evict += 1
    u = O.rollout(sp, 11, 3, algo=1, cfg0=cfg)
    assert int(r.totals["n_preempt"]) == n_evict
    assert n_evict <= 0.4 * int(u.totals["n_preempt"])
    assert int(r.totals["n_completed"]) == int(u.totals["n_completed"])


def test_restricted_preemption_equals_edf_ss_when_nothing_ever_waits():
    # sparse arrivals (no two jobs overlap): both variants place every job on the slowest slice that meets its deadline
    sp = tiny_params()
    rows = [(1000 * i, 0, 5 + i % 7, 1000 * i + 40 + 13 * (i % 5)) for i in range(60)]
    a = O.rollout(sp, 0, 0, algo=4, cfg0=2, jobs=O.make_jobs(rows), trace_cap=1024)
    b = O.rollout(sp, 0, 0, algo=1, cfg0=2, jobs=O.make_jobs(rows), trace_cap=1024)
    assert a.trace.tobytes() == b.trace.tobytes() and a.totals.tobytes() == b.totals.tobytes()


def test_restricted_preemption_with_repartitions_keeps_the_invariants():
    rng = np.random.default_rng(5)
    table = rng.integers(0, 12, size=(24, 4)).astype(np.uint8)
    sp, r = _restricted_day(1, 4, table=table)
    assert int(r.totals["n_repart"]) > 10 and int(r.totals["n_jobs"]) == int(r.totals["n_completed"]) + int(r.totals["n_dropped"])


def test_event_driven_decisions_with_a_load_blind_table_equal_hourly_decisions():
    # reading #27: a table whose four load buckets agree gives the same action at every event of an epoch as at its
    # start, so the event-driven run must be the hourly run, event for event
    import dataclasses
    wl = W.config_c3(4)
    for e in range(3):
        a = O.rollout(wl.params, 3, e, algo=1, cfg0=int(wl.cfg0[e]), policy=W.POLICY_TABLE, table=wl.table[e], trace_cap=100000)
        b = O.rollout(dataclasses.replace(wl.params, decide_on_events=1), 3, e, algo=1, cfg0=int(wl.cfg0[e]), policy=W.POLICY_TABLE,
                      table=wl.table[e], trace_cap=100000)
        assert int(a.totals["n_repart"]) == 2 and a.trace.tobytes() == b.trace.tobytes() and a.recs.tobytes() == b.recs.tobytes()


@pytest.mark.parametrize("algo", [1, 2, 4])
def test_event_driven_decisions_keep_the_invariants(algo):
    import dataclasses
    wl = W.config_c3(4)
    sp = dataclasses.replace(wl.params, decide_on_events=1, repart_downtime_s=4, repart_energy_mj=1000)
    table = np.random.default_rng(algo).integers(0, 12, size=(24, 4)).astype(np.uint8)
    r = O.rollout(sp, 9, 1, algo=algo, cfg0=3, policy=W.POLICY_TABLE, table=table, trace_cap=400000)
    assert int(r.totals["status"]) == 0 and int(r.totals["n_repart"]) > 100       # the load crosses bucket borders all day
    trace_check.check_against_records(sp, 3, r.trace, r.recs, r.totals)
    rep = [int(ev["t"]) for ev in r.trace if ev["type"] == 8 and ev["t"] % 3600 != 0]
    job_ticks = {int(ev["t"]) for ev in r.trace if ev["type"] in (1, 2, 5)}
    assert rep and all(t in job_ticks for t in rep)                                # only where a job arrived or completed


@pytest.mark.parametrize("cfg", [0, 4])
def test_uniform_slice_configs_make_variants_coincide(cfg):
    # "configurations 1 and 5 ... the EDF variants produce the same value, as do the LLF variants"
    wl = W.config_c2(8)
    for e in range(8):
        tr = [O.rollout(wl.params, wl.seed, e, algo=a, cfg0=cfg, trace_cap=60000) for a in range(4)]
        assert trace_tuple(tr[0].trace) == trace_tuple(tr[1].trace)
        assert trace_tuple(tr[2].trace) == trace_tuple(tr[3].trace)
        assert int(tr[0].totals["trace_hash"]) == int(tr[1].totals["trace_hash"])
        assert int(tr[2].totals["trace_hash"]) == int(tr[3].totals["trace_hash"])


def test_variants_differ_on_mixed_configs():
    wl = W.config_c2(4)
    h = {a: int(O.rollout(wl.params, wl.seed, 0, algo=a, cfg0=2).totals["trace_hash"]) for a in range(4)}
    assert len(set(h.values())) == 4


def test_single_machine_energy_closed_form():
    # cfg 1, work-conserving single machine: E = P_idle * T + (P_busy - P_idle) * sum dur7, for every algorithm
    wl = W.config_c2(4)
    sp = wl.params
    for e in range(4):
        for algo in range(4):
            r = O.rollout(sp, wl.seed, e, algo=algo, cfg0=0, trace_cap=60000)
            arrive = {int(ev["job"]): ev for ev in r.trace if ev["type"] == 1}
            first_start = {}
            for ev in r.trace:
                if ev["type"] == 3 and int(ev["job"]) not in first_start:
                    first_start[int(ev["job"])] = int(ev["value"])
            busy_s = sum(v // 840 for v in first_start.values())        # work = dur7 * 840
            assert all(v % 840 == 0 for v in first_start.values())
            T = max(86400, int(r.totals["t_end"]))
            assert int(r.totals["energy_mj"]) == 60000 * T + 188243 * busy_s
            assert int(r.totals["busy_unit_s"]) == 7 * busy_s
            assert len(arrive) == len(first_start)


def test_sparse_arrivals_closed_form():
    # jobs far apart never overlap: EDF-FS finishes at arr + rd(largest slice); EDF-SS at arr + rd(slowest feasible)
    sp = tiny_params()
    rows, t = [], 100
    rng = np.random.default_rng(5)
    for i in range(40):
        dur7 = int(rng.integers(2, 60))
        slack = float(rng.uniform(1.2, 9.0))
        rows.append((t, 0, dur7, t + max(1, int(dur7 * slack))))
        t += 1000
    jobs = O.make_jobs(rows)
    for cfg in range(12):
        sizes = sorted(int(g) for g in sp.size_at_slot[cfg] if g)
        idle = sum(int(sp.p_idle_mw[W.SIZE_INDEX[g]]) for g in sizes)
        dyn = {g: int(sp.p_busy_mw[W.SIZE_INDEX[g]] - sp.p_idle_mw[W.SIZE_INDEX[g]]) for g in sizes}
        for algo in (0, 1):
            r = O.rollout(sp, 0, 0, algo=algo, cfg0=cfg, jobs=jobs, trace_cap=1000)
            comp = completions(r.trace)
            e_dyn = 0
            for i, (arr, _, dur7, due) in enumerate(rows):
                work = dur7 * 840
                rd = {g: -(-work // (120 * g)) for g in sizes}
                g_fast = max(sizes)
                if algo == 1:
                    feas = [g for g in sizes if arr + rd[g] <= due]
                    g_use = min(feas) if feas else g_fast
                else:
                    g_use = g_fast
                assert comp[i] == arr + rd[g_use], (cfg, algo, i)
                e_dyn += dyn[g_use] * rd[g_use]
            assert int(r.totals["energy_mj"]) == idle * 86400 + e_dyn
            assert int(r.totals["n_preempt"]) == 0


# ------------------------------------------------------------------------------------- brute force, single machine
def _lmax(order, rows):
    t, worst = 0, -10 ** 9
    for i in order:
        t += rows[i][2]
        worst = max(worst, t - rows[i][3])
    return worst


def test_edd_minimises_max_lateness_all_released_at_zero():
    # Jackson's rule: all jobs released at 0 on one machine -> EDF order minimises L_max (brute force over <= 5! orders)
    rng = np.random.default_rng(17)
    sp = tiny_params()
    for trial in range(40):
        n = int(rng.integers(2, 6))
        rows = [(0, 0, int(rng.integers(1, 9)), int(rng.integers(1, 30))) for _ in range(n)]
        best = min(_lmax(o, rows) for o in itertools.permutations(range(n)))
        for algo in (0, 1):
            r = O.rollout(sp, 0, 0, algo=algo, cfg0=0, jobs=O.make_jobs(rows), trace_cap=200)
            comp = completions(r.trace)
            got = max(comp[i] - rows[i][3] for i in range(n))
            assert got == best, (rows, got, best)
            assert int(r.totals["n_preempt"]) == 0
            assert int(r.totals["tardiness_s"]) == sum(max(comp[i] - rows[i][3], 0) for i in range(n))


def _best_lmax_preemptive(rows, horizon):
    """Brute force over every unit-slot schedule of one machine (release dates, preemption allowed)."""
    n = len(rows)
    best = [10 ** 9]
    rem0 = [r[2] for r in rows]

    def rec(t, rem, comp):
        if all(x == 0 for x in rem):
            best[0] = min(best[0], max(comp[i] - rows[i][3] for i in range(n)))
            return
        if t >= horizon:
            return
        ready = [i for i in range(n) if rem[i] > 0 and rows[i][0] <= t]
        if not ready:
            rec(t + 1, rem, comp)
            return
        for i in ready:                       # idling with a ready job is never better for L_max
            rem[i] -= 1
            old = comp[i]
            if rem[i] == 0:
                comp[i] = t + 1
            rec(t + 1, rem, comp)
            comp[i] = old
            rem[i] += 1

    rec(0, rem0, [0] * n)
    return best[0]


def test_preemptive_edf_minimises_max_lateness_with_release_dates():
    # Horn: preemptive EDF minimises L_max on one machine with release dates; total work <= 10 ticks
    rng = np.random.default_rng(23)
    sp = tiny_params()
    for trial in range(25):
        n = int(rng.integers(2, 5))
        durs = [int(rng.integers(1, 4)) for _ in range(n)]
        while sum(durs) > 10:
            durs[int(np.argmax(durs))] -= 1
        rows = sorted([(int(rng.integers(0, 6)), 0, d, 0) for d in durs])
        rows = [(a, c, d, a + int(rng.integers(1, 9))) for (a, c, d, _) in rows]
        best = _best_lmax_preemptive(rows, 6 + 10)
        r = O.rollout(sp, 0, 0, algo=0, cfg0=0, jobs=O.make_jobs(rows), trace_cap=200)
        comp = completions(r.trace)
        got = max(comp[i] - rows[i][3] for i in range(n))
        assert got == best, (rows, got, best)
        if best <= 0:
            assert int(r.totals["tardiness_s"]) == 0


def test_queue_cap_drops_and_counts():
    sp = tiny_params(cap=256)
    rows = [(5, 0, 100, 100000)] * 300                  # 300 simultaneous arrivals, cap 256 jobs in system
    r = O.rollout(sp, 0, 0, algo=0, cfg0=0, jobs=O.make_jobs(rows), trace_cap=2000)
    assert int(r.totals["n_jobs"]) == 300 and int(r.totals["n_dropped"]) == 44 and int(r.totals["n_completed"]) == 256
    drops = [int(ev["job"]) for ev in r.trace if ev["type"] == 2]
    assert drops == list(range(256, 300))
    assert int(r.totals["n_sys_max"]) == 256
    assert int(r.recs[0]["n_dropped"]) == 44
    trace_check.check_against_records(sp, 0, r.trace, r.recs, r.totals)


def test_truncation_flag():
    sp = tiny_params(t_limit_s=90000)
    rows = [(0, 0, 100000, 50)]                         # needs 100000 s on 7g; horizon 90000
    r = O.rollout(sp, 0, 0, algo=0, cfg0=0, jobs=O.make_jobs(rows), trace_cap=100)
    assert int(r.totals["status"]) & O.ST_TRUNCATED
    assert int(r.totals["n_completed"]) == 0 and int(r.totals["t_end"]) == 90000
    assert int(r.totals["energy_mj"]) == 248243 * 90000


def test_bad_action_is_stay():
    sp = tiny_params()
    env = O.Env(sp, 0, 0, jobs=O.make_jobs([(10, 0, 5, 100)]), trace_cap=100)
    env.reset(algo=0, cfg0=3)
    _, _, dE, _, rec = env.step(200)
    assert int(rec[0]["status"]) & O.ST_BAD_ACTION and int(rec[0]["cfg"]) == 3 and int(rec[0]["repartitioned"]) == 0


def test_step_composition_equals_rollout():
    wl = W.config_c3(3)
    sp = wl.params
    for e in range(3):
        r = O.rollout(sp, wl.seed, e, algo=1, cfg0=int(wl.cfg0[e]), policy=W.POLICY_TABLE, table=wl.table[e], want_states=True)
        env = O.Env(sp, wl.seed, e)
        x = env.reset(algo=1, cfg0=int(wl.cfg0[e]))
        assert np.array_equal(x, r.states[0])
        for k in range(24):
            x, rew, dE, dT, rec = env.step(int(r.actions[k]))
            assert np.array_equal(x, r.states[k + 1]) and rew == r.rewards[k]
            assert rec[0].tobytes() == r.recs[k].tobytes()
        assert env.totals().tobytes() == r.totals.tobytes()
        with pytest.raises(RuntimeError):
            env.step(0)
