"""GPU parity: the CUDA path (through the C ABI) vs the CPU oracle, element by element, on the same seeded inputs.

Bar (north_star): BIT-EXACT on every event trace and integer objective component; the fp32 state vector is exact by
construction (small integers times powers of two); Q-values and rewards are compared bit-for-bit as well (fixed-order
fmaf / two products and an add), which is stricter than the 1e-4 relative tolerance north_star allows.
"""
import concurrent.futures as cf
import dataclasses
import os

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
import trace_check
from util import CAP3, LINEAR, SUB05, golden, tiny_params

pytestmark = pytest.mark.gpu

B = None


# every test runs on both rollout kernels: 8-lane warp tiles and one thread per environment (mig_sim_set_tile)
@pytest.fixture(scope="module", autouse=True, params=[8, 1], ids=["tile8", "thread"])
def _binding(request):
    global B
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_25082_b200 import binding
    B = binding
    B.DEFAULT_TILE = request.param
    yield
    B.DEFAULT_TILE = 0


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ------------------------------------------------------------------------------------------------ oracle side
def _oracle_env(args):
    wl_name, n_envs, e, want_trace, overrides = args
    wl = W.CONFIGS[wl_name](n_envs)
    sp = wl.params
    r = O.rollout(sp, wl.seed, e + sp.env_offset, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy,
                  table=None if wl.table is None else wl.table[e], qnet=wl.qnet, epsilon=wl.epsilon,
                  trace_cap=600000 if want_trace else 0, want_states=True)
    return e, r.recs, r.totals, (r.trace if want_trace else None), r.states, r.actions, r.rewards


_ORACLE_CACHE = {}


def oracle_many(wl_name, n_envs, envs, want_trace=False):
    key = (wl_name, n_envs, tuple(int(e) for e in envs), want_trace)          # the oracle's answers serve both kernels
    if key not in _ORACLE_CACHE:
        _ORACLE_CACHE[key] = _oracle_many(wl_name, n_envs, envs, want_trace)
    return _ORACLE_CACHE[key]


def _oracle_many(wl_name, n_envs, envs, want_trace=False):
    args = [(wl_name, n_envs, int(e), want_trace, None) for e in envs]
    workers = min(len(args), os.cpu_count() or 1)
    if workers <= 1:
        return [_oracle_env(a) for a in args]
    with cf.ProcessPoolExecutor(workers) as ex:
        return list(ex.map(_oracle_env, args, chunksize=max(1, len(args) // (4 * workers))))


def _oracle_bulk_chunk(args):
    wl_name, n_envs, lo, hi = args
    wl = W.CONFIGS[wl_name](n_envs)
    ph = O.ParamsHolder(wl.params)
    qh = O.QNetHolder(wl.qnet) if wl.qnet is not None else None
    recs = np.zeros((ph.sp.n_epochs + 1, hi - lo), dtype=O.REC_DTYPE)
    tots = np.zeros(hi - lo, dtype=O.TOTALS_DTYPE)
    for e in range(lo, hi):
        r = O.rollout(ph, wl.seed, e + wl.params.env_offset, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy,
                      table=None if wl.table is None else wl.table[e], qnet=qh, epsilon=wl.epsilon)
        recs[:, e - lo] = r.recs
        tots[e - lo] = r.totals
    return lo, hi, recs, tots


def oracle_bulk(wl_name, n_envs):
    """EVERY env-day of the workload on the oracle (records, totals, trace hash), all host cores; cached for both kernels."""
    key = ("bulk", wl_name, n_envs)
    if key not in _ORACLE_CACHE:
        ne = W.CONFIGS[wl_name](1).params.n_epochs
        recs = np.zeros((ne + 1, n_envs), dtype=O.REC_DTYPE)
        tots = np.zeros(n_envs, dtype=O.TOTALS_DTYPE)
        workers = os.cpu_count() or 1
        step = max(1, min(256, n_envs // (4 * workers)))
        tasks = [(wl_name, n_envs, lo, min(n_envs, lo + step)) for lo in range(0, n_envs, step)]
        with cf.ProcessPoolExecutor(workers) as ex:
            for lo, hi, r, t in ex.map(_oracle_bulk_chunk, tasks):
                recs[:, lo:hi] = r
                tots[lo:hi] = t
        _ORACLE_CACHE[key] = (recs, tots)
    return _ORACLE_CACHE[key]


def gpu_rollout(wl, sim=None, qnet=None):
    sim = sim or B.MigSim(wl.params, wl.n_envs, wl.seed)
    recs, totals = sim.alloc_recs(), sim.alloc_totals()
    sim.reset(0, dev(wl.algo), dev(wl.cfg0))
    table = None if wl.table is None else dev(wl.table)
    if wl.policy == W.POLICY_DQN and qnet is None:
        qnet = B.QNet(wl.qnet)
    sim.rollout(wl.policy, table=table, qnet=qnet, epsilon=wl.epsilon, recs_out=recs, totals_out=totals)
    torch.cuda.synchronize()
    return sim, B.recs_to_numpy(recs), B.totals_to_numpy(totals), table


def assert_same_records(g_recs, g_tot, o_recs, o_tot, tag):
    assert g_tot.tobytes() == o_tot.tobytes(), "%s totals differ:\n gpu %s\n orc %s" % (tag, g_tot, o_tot)
    for k in range(len(o_recs)):
        assert g_recs[k].tobytes() == o_recs[k].tobytes(), "%s record %d differs:\n gpu %s\n orc %s" % (tag, k, g_recs[k], o_recs[k])


def compare_workload(name, n_envs, trace_envs):
    """Records, totals and trace hash of EVERY env against the oracle; full event traces for trace_envs."""
    wl = W.CONFIGS[name](n_envs)
    sim, recs, totals, table = gpu_rollout(wl)
    assert np.all(totals["status"] == 0)
    o_recs_all, o_tot_all = oracle_bulk(name, n_envs)
    if totals.tobytes() != o_tot_all.tobytes() or recs.tobytes() != o_recs_all.tobytes():
        bad = [e for e in range(n_envs) if totals[e].tobytes() != o_tot_all[e].tobytes() or recs[:, e].tobytes() != o_recs_all[:, e].tobytes()]
        e = bad[0]
        assert_same_records(recs[:, e], totals[e], o_recs_all[:, e], o_tot_all[e], "%s: %d of %d envs differ; env %d" % (name, len(bad), n_envs, e))
    # full event trace for a subset (DQN: replay the actions the rollout took = the records' cfg)
    for e, o_recs, o_tot, o_trace, _, o_act, _ in oracle_many(name, n_envs, trace_envs, want_trace=True):
        if wl.policy == W.POLICY_DQN:
            ev, tot = sim.debug_trace(e, actions=dev(recs[:24, e]["cfg"].astype(np.uint8)))
        else:
            ev, tot = sim.debug_trace(e, policy=wl.policy, table=table)
        assert len(ev) == len(o_trace), "%s env %d: %d events vs %d" % (name, e, len(ev), len(o_trace))
        if ev.tobytes() != o_trace.tobytes():
            i = int(np.nonzero(ev != o_trace)[0][0])
            raise AssertionError("%s env %d: first differing event %d:\n gpu %s\n orc %s" % (name, e, i, ev[max(0, i - 3):i + 2], o_trace[max(0, i - 3):i + 2]))
        assert tot.tobytes() == o_tot.tobytes()
        trace_check.check_against_records(wl.params, int(wl.cfg0[e]), ev, recs[:, e], totals[e])
    sim.close()
    return totals


# ------------------------------------------------------------------------------------------------ BASELINE configs
def test_c1_full_trace():
    compare_workload("C1", 1, [0])


def test_c2_all_envs_all_algorithms_all_configs():
    tot = compare_workload("C2", 1024, range(0, 1024, 16))
    assert tot["n_jobs"].sum() > 1024 * 1900


def test_c3_twice_daily_repartitioning():
    tot = compare_workload("C3", 4096, range(0, 4096, 64))
    assert np.all(tot["n_repart"] == 2)


def test_c4_dqn_driven():
    tot = compare_workload("C4", 8192, range(0, 8192, 128))
    assert tot["n_repart"].mean() > 5


def test_c5_full_size_every_env():
    # BASELINE's full size in the launch configuration bench.py times: all 65 536 env-days (about 10^9 job-events) are
    # simulated by the oracle on the host cores and compared record by record ("C5 full parity ... run once")
    tot = compare_workload("C5", 65536, range(0, 65536, 4096))
    # properties that hold at any size
    assert np.all(tot["n_jobs"] == tot["n_completed"] + tot["n_dropped"])
    assert abs(tot["n_jobs"].mean() - 8000) < 8000 * 0.01


# ------------------------------------------------------------------------------------------------ hand-worked schedules on the GPU
G = golden("handworked.json")


def gpu_script(sp, rows, algo, cfg, n_envs=1, actions=None, cap_events=4096):
    sim = B.MigSim(sp, n_envs, 0)
    jobs = O.make_jobs(rows).astype(B.JOB_DTYPE)
    sim.debug_set_jobs(jobs)
    sim.reset(0, dev(np.full(n_envs, algo, np.uint8)), dev(np.full(n_envs, cfg, np.uint8)))
    ev, tot = sim.debug_trace(0, actions=None if actions is None else dev(np.asarray(actions, np.uint8)), cap_events=cap_events)
    sim.close()
    return ev, tot


@pytest.mark.parametrize("case,algos,speeds,kw", [
    ("A", [0, 1, 2, 3], (LINEAR,), dict(crit_laxity_s=1)),
    ("B", [0, 1], (LINEAR,), {}),
    ("C", [0, 1], (LINEAR,), {}),
    ("E", [0, 1, 2, 3], (LINEAR,), dict(crit_laxity_s=5, crit_max=3)),
    ("F", [0, 2, 3], (LINEAR, SUB05), dict(crit_laxity_s=1)),
    ("G", [0, 1, 2, 3], (CAP3,), {}),
    ("H", [4, 1], (LINEAR,), {}),
    ("I", [4, 1], (LINEAR,), {}),
])
def test_handworked_schedules_trace_equal(case, algos, speeds, kw):
    g = G[case]
    sp = tiny_params(speeds=speeds, **kw)
    for algo in algos:
        ev, tot = gpu_script(sp, g["jobs"], algo, g["cfg"])
        r = O.rollout(sp, 0, 0, algo=algo, cfg0=g["cfg"], jobs=O.make_jobs(g["jobs"]), trace_cap=256)
        assert ev.tobytes() == r.trace.tobytes(), (case, algo, ev, r.trace)
        assert tot.tobytes() == r.totals.tobytes()


def test_handworked_values_direct():
    # the GPU against the hand-computed numbers themselves (not via the oracle)
    g = G["B"]
    sp = tiny_params()
    for name, algo in (("EDF-FS", 0), ("EDF-SS", 1)):
        ev, tot = gpu_script(sp, g["jobs"], algo, g["cfg"])
        comp = {int(e["job"]): int(e["t"]) for e in ev if e["type"] == 5}
        assert comp == {int(k): v for k, v in g[name]["completion"].items()}
        assert int(tot["energy_mj"]) == g["idle_mw"] * 86400 + g[name]["dyn_energy_mj"]
    g = G["D"]
    sp = tiny_params(repart_downtime_s=g["downtime_s"], repart_energy_mj=g["repart_energy_mj"])
    acts = [g["cfg0"]] + [g["action_epoch1"]] * 23
    ev, tot = gpu_script(sp, g["jobs"], g["algo"], g["cfg0"], actions=acts)
    comp = {int(e["job"]): int(e["t"]) for e in ev if e["type"] == 5}
    assert comp == {int(k): v for k, v in g["completion"].items()}
    assert int(tot["n_repart"]) == 1 and int(tot["tardiness_s"]) == 0
    assert int(tot["energy_mj"]) == g["epoch0_energy_mj"] + g["epoch1_energy_mj"] + 22 * 85000 * 3600


# ------------------------------------------------------------------------------------------------ step API, states, rewards
@pytest.mark.parametrize("name,n", [("C3", 96), ("C4", 96), ("C2", 96)])
def test_step_equals_rollout_and_oracle_states(name, n):
    wl = W.CONFIGS[name](n)
    res = {e: r for e, *r in oracle_many(name, n, range(n))}
    sim = B.MigSim(wl.params, n, wl.seed)
    state = sim.alloc_state()
    sim.reset(0, dev(wl.algo), dev(wl.cfg0), state_out=state)
    s0 = state.cpu().numpy()
    for e in range(n):
        assert np.array_equal(s0[e], res[e][3][0])
    reward = torch.zeros(n, dtype=torch.float32, device="cuda")
    dE = torch.zeros(n, dtype=torch.int64, device="cuda")
    dT = torch.zeros(n, dtype=torch.int64, device="cuda")
    rec = torch.zeros((n, 64), dtype=torch.uint8, device="cuda")
    drain = torch.zeros((n, 64), dtype=torch.uint8, device="cuda")
    for k in range(24):
        act = np.array([res[e][4][k] for e in range(n)], dtype=np.uint8)       # the oracle's actions (teacher forcing)
        sim.step(dev(act), state_out=state, reward_out=reward, energy_out=dE, tard_out=dT, rec_out=rec, drain_rec_out=drain)
        torch.cuda.synchronize()
        s, rw, recs = state.cpu().numpy(), reward.cpu().numpy(), B.recs_to_numpy(rec)
        for e in range(n):
            o_recs, o_tot, _, o_states, o_act, o_rew = res[e]
            assert recs[e].tobytes() == o_recs[k].tobytes(), (name, e, k, recs[e], o_recs[k])
            assert np.array_equal(s[e], o_states[k + 1]), (name, e, k, s[e], o_states[k + 1])
            assert rw[e].tobytes() == np.float32(o_rew[k]).tobytes(), (name, e, k)
            extra = int(o_recs[24]["energy_mj"]) if k == 23 else 0
            assert int(dE[e]) == int(o_recs[k]["energy_mj"]) + extra
    dr = B.recs_to_numpy(drain)
    tot = sim.alloc_totals()
    sim.totals(tot)
    tot = B.totals_to_numpy(tot)
    for e in range(n):
        assert dr[e].tobytes() == res[e][0][24].tobytes()
        assert tot[e].tobytes() == res[e][1].tobytes()
    with pytest.raises(B.MigError) as ei:
        sim.step(dev(np.zeros(n, np.uint8)))
    assert ei.value.code == B.MIG_ESTATE
    sim.close()


def test_partial_steps_then_rollout():
    wl = W.config_c3(64)
    _, recs_ref, tot_ref, table = gpu_rollout(wl)
    sim = B.MigSim(wl.params, 64, wl.seed)
    sim.reset(0, dev(wl.algo), dev(wl.cfg0))
    for k in range(7):
        sim.step(dev(recs_ref[k]["cfg"].astype(np.uint8)))
    recs, tot = sim.alloc_recs(), sim.alloc_totals()
    sim.rollout(W.POLICY_TABLE, table=table, recs_out=recs, totals_out=tot)
    torch.cuda.synchronize()
    assert B.totals_to_numpy(tot).tobytes() == tot_ref.tobytes()
    assert B.recs_to_numpy(recs)[7:].tobytes() == recs_ref[7:].tobytes()
    sim.close()


def test_rollout_host_matches_device_rollout():
    for name, n in (("C3", 128), ("C4", 128)):
        wl = W.CONFIGS[name](n)
        _, recs_ref, tot_ref, _ = gpu_rollout(wl)
        sim = B.MigSim(wl.params, n, wl.seed)
        q = B.QNet(wl.qnet) if wl.qnet is not None else None
        tot = np.zeros(n, dtype=B.TOTALS_DTYPE)
        recs = np.zeros((25, n), dtype=B.REC_DTYPE)
        sim.rollout_host(0, wl.algo, wl.cfg0, wl.policy, wl.table, q, wl.epsilon, recs, tot)
        assert tot.tobytes() == tot_ref.tobytes() and recs.tobytes() == recs_ref.tobytes()
        # result buffers in pinned, mapped host memory: the kernels write them directly (no copy after the launch)
        tot2, recs2 = np.zeros(n, dtype=B.TOTALS_DTYPE), np.zeros((25, n), dtype=B.REC_DTYPE)
        rt = torch.cuda.cudart()
        for a in (tot2, recs2):
            assert int(rt.cudaHostRegister(a.ctypes.data, a.nbytes, 0)) == 0
        try:
            sim.rollout_host(0, wl.algo, wl.cfg0, wl.policy, wl.table, q, wl.epsilon, recs2, tot2)
            assert tot2.tobytes() == tot_ref.tobytes() and recs2.tobytes() == recs_ref.tobytes()
            recs2[:] = 0                                    # records mapped, totals not
            tot3 = np.zeros(n, dtype=B.TOTALS_DTYPE)
            sim.rollout_host(0, wl.algo, wl.cfg0, wl.policy, wl.table, q, wl.epsilon, recs2, tot3)
            assert tot3.tobytes() == tot_ref.tobytes() and recs2.tobytes() == recs_ref.tobytes()
        finally:
            for a in (tot2, recs2):
                rt.cudaHostUnregister(a.ctypes.data)
        sim.close()


def test_env_base_sharding_is_placement_invariant():
    import dataclasses
    wl = W.config_c3(64)
    _, recs_ref, tot_ref, _ = gpu_rollout(wl)
    for lo, hi in (W.shard_range(64, 0, 2), W.shard_range(64, 1, 2)):
        sp = dataclasses.replace(wl.params, env_offset=lo)
        sim = B.MigSim(sp, hi - lo, wl.seed)
        recs, tot = sim.alloc_recs(), sim.alloc_totals()
        sim.reset(0, dev(wl.algo[lo:hi]), dev(wl.cfg0[lo:hi]))
        sim.rollout(wl.policy, table=dev(wl.table[lo:hi]), recs_out=recs, totals_out=tot)
        torch.cuda.synchronize()
        assert B.totals_to_numpy(tot).tobytes() == tot_ref[lo:hi].tobytes()
        sim.close()


def test_both_kernel_bodies_give_the_same_days():
    # The thread-per-environment kernel has two bodies: one with the laxity algorithms compiled out, taken when the whole
    # batch runs deadline-keyed algorithms (EDF-FS, EDF-SS, restricted EDF-SS), and the generic one.  The same 96 envs are
    # run alone (short body) and next to one LLF env (generic body); the step API and the rollout are both exercised.
    if B.DEFAULT_TILE not in (0, 1):
        pytest.skip("thread-per-environment kernel only")
    n = 96
    wl = W.config_c3(n + 1)
    algo = np.concatenate([np.array([0, 1, 4] * (n // 3), np.uint8), [2]]).astype(np.uint8)      # the last env runs LLF
    out = []
    for m in (n, n + 1):
        sim = B.MigSim(wl.params, m, wl.seed)
        recs, tot = sim.alloc_recs(), sim.alloc_totals()
        sim.reset(0, dev(algo[:m]), dev(wl.cfg0[:m]))
        acts = [dev(wl.table[:m, k, 0].copy()) for k in range(3)]
        for k in range(3):                                     # three epochs through mig_sim_step, the rest through the rollout
            sim.step(acts[k])
        sim.rollout(wl.policy, table=dev(wl.table[:m]), recs_out=recs, totals_out=tot)
        torch.cuda.synchronize()
        out.append((B.recs_to_numpy(recs)[3:, :n].copy(), B.totals_to_numpy(tot)[:n].copy()))
        sim.close()
    assert out[0][1].tobytes() == out[1][1].tobytes() and out[0][0].tobytes() == out[1][0].tobytes()
    for e in (0, 1, 2, 50):
        r = O.rollout(wl.params, wl.seed, e, algo=int(algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy, table=wl.table[e])
        assert out[0][1][e].tobytes() == r.totals.tobytes()


def _oracle_custom(args):
    sp, seed, e, algo, cfg0, table = args
    r = O.rollout(sp, seed, e, algo=algo, cfg0=cfg0, policy=W.POLICY_TABLE, table=table, trace_cap=400000, want_states=True)
    return e, r.recs, r.totals, r.trace, r.states


@pytest.mark.parametrize("downtime,theta", [(60, 60), (0, 5), (1800, 600)])
def test_hourly_random_repartitions_all_algorithms(downtime, theta):
    # every env repartitions to a random configuration every hour (a different one per load bucket), algorithms cycle
    # over EDF-FS / EDF-SS / LLF / LALF: repartition with requeue, downtime, re-keyed laxities and critical-laxity events
    import dataclasses
    n = 64
    base = W.config_c3(n)
    sp = dataclasses.replace(base.params, repart_downtime_s=downtime, crit_laxity_s=theta)
    rng = np.random.default_rng(downtime + theta)
    table = rng.integers(0, 12, size=(n, 24, 4)).astype(np.uint8)
    algo = (np.arange(n) % 5).astype(np.uint8)               # EDF-FS, EDF-SS, LLF, LALF, EDF-SS with restricted preemption
    cfg0 = rng.integers(0, 12, size=n).astype(np.uint8)
    sim = B.MigSim(sp, n, 77)
    recs, tot = sim.alloc_recs(), sim.alloc_totals()
    state = sim.alloc_state()
    d_table = dev(table)
    sim.reset(0, dev(algo), dev(cfg0))
    sim.rollout(W.POLICY_TABLE, table=d_table, recs_out=recs, totals_out=tot)
    sim.totals(tot)
    torch.cuda.synchronize()
    g_recs, g_tot = B.recs_to_numpy(recs), B.totals_to_numpy(tot)
    with cf.ProcessPoolExecutor(min(n, os.cpu_count() or 1)) as ex:
        res = list(ex.map(_oracle_custom, [(sp, 77, e, int(algo[e]), int(cfg0[e]), table[e]) for e in range(n)]))
    assert g_tot["n_repart"].min() > 10 and (theta > 60 or g_tot["n_crit"][2::5].sum() > 0)
    for e, o_recs, o_tot, o_trace, o_states in res:
        assert_same_records(g_recs[:, e], g_tot[e], o_recs, o_tot, "env %d algo %d" % (e, algo[e]))
    for e, o_recs, o_tot, o_trace, o_states in res[:16]:
        ev, t1 = sim.debug_trace(e, policy=W.POLICY_TABLE, table=d_table, cap_events=400000)
        assert len(ev) == len(o_trace) and ev.tobytes() == o_trace.tobytes(), "env %d" % e
    # the same day step by step with the actions the rollout took: states after every epoch
    sim.reset(0, dev(algo), dev(cfg0), state_out=state)
    for k in range(24):
        sim.step(dev(g_recs[k]["cfg"].astype(np.uint8)), state_out=state)
        torch.cuda.synchronize()
        s_k = state.cpu().numpy()
        for e, o_recs, o_tot, o_trace, o_states in res:
            assert np.array_equal(s_k[e], o_states[k + 1]), (e, k)
    sim.close()


@pytest.mark.parametrize("downtime", [4, 60])
def test_event_driven_table_decisions(downtime):
    # PAPER.md:L212 / reading #27: the tabulated policy is looked up again after every tick with an arrival or a
    # completion; random bucket-dependent tables make the configuration follow the load all day, all five algorithms
    import dataclasses
    n = 60
    base = W.config_c3(n)
    sp = dataclasses.replace(base.params, repart_downtime_s=downtime, repart_energy_mj=1000, decide_on_events=1)
    rng = np.random.default_rng(downtime)
    table = rng.integers(0, 12, size=(n, 24, 4)).astype(np.uint8)
    table[::7] = table[::7, :, :1]                                   # some load-blind tables: decisions stay hourly
    algo = (np.arange(n) % 5).astype(np.uint8)
    cfg0 = rng.integers(0, 12, size=n).astype(np.uint8)
    sim = B.MigSim(sp, n, 55)
    recs, tot = sim.alloc_recs(), sim.alloc_totals()
    d_table = dev(table)
    sim.reset(0, dev(algo), dev(cfg0))
    sim.rollout(W.POLICY_TABLE, table=d_table, recs_out=recs, totals_out=tot)
    torch.cuda.synchronize()
    g_recs, g_tot = B.recs_to_numpy(recs), B.totals_to_numpy(tot)
    with cf.ProcessPoolExecutor(min(n, os.cpu_count() or 1)) as ex:
        res = list(ex.map(_oracle_custom, [(sp, 55, e, int(algo[e]), int(cfg0[e]), table[e]) for e in range(n)]))
    assert np.median(g_tot["n_repart"]) > 100 and g_tot["n_repart"][::7].max() <= 24
    for e, o_recs, o_tot, o_trace, o_states in res:
        assert_same_records(g_recs[:, e], g_tot[e], o_recs, o_tot, "env %d algo %d" % (e, algo[e]))
    for e, o_recs, o_tot, o_trace, o_states in res[:10]:
        ev, t1 = sim.debug_trace(e, policy=W.POLICY_TABLE, table=d_table, cap_events=400000)
        assert len(ev) == len(o_trace) and ev.tobytes() == o_trace.tobytes(), "env %d" % e
    sim.close()


def test_event_driven_handworked_J():
    import dataclasses
    g = G["J"]
    sp = dataclasses.replace(tiny_params(repart_downtime_s=g["downtime_s"], repart_energy_mj=g["repart_energy_mj"]), decide_on_events=1)
    table = np.zeros((1, 24, 4), np.uint8)
    table[:, :, 0] = g["table"]["bucket0"]; table[:, :, 1:] = g["table"]["bucket1_3"]
    sim = B.MigSim(sp, 1, 0)
    sim.debug_set_jobs(O.make_jobs(g["jobs"]).astype(B.JOB_DTYPE))
    sim.reset(0, dev(np.array([g["algo"]], np.uint8)), dev(np.array([g["cfg0"]], np.uint8)))
    ev, tot = sim.debug_trace(0, policy=W.POLICY_TABLE, table=dev(table), cap_events=64)
    assert [[int(e["t"]), int(e["type"]), int(e["slot"])] for e in ev] == [[t, {"ARRIVE": 1, "START": 3, "PREEMPT": 4, "COMPLETE": 5, "SLICE_UP": 7, "REPART": 8}[nm], sl] for t, nm, jb, sl in g["events"]]
    assert int(tot["n_repart"]) == g["n_repart"]
    r = O.rollout(sp, 0, 0, algo=g["algo"], cfg0=g["cfg0"], policy=W.POLICY_TABLE, table=table[0], jobs=O.make_jobs(g["jobs"]), trace_cap=64)
    assert ev.tobytes() == r.trace.tobytes() and tot.tobytes() == r.totals.tobytes()
    sim.close()


def _oracle_static(args):
    sp, seed, e, algo, cfg0, want_trace = args
    r = O.rollout(sp, seed, e, algo=algo, cfg0=cfg0, trace_cap=400000 if want_trace else 0)
    return e, r.recs, r.totals, r.trace if want_trace else None


@pytest.mark.parametrize("name,seed", [("C2", 21), ("C5", 22)])
def test_restricted_preemption_static_configs(name, seed):
    # EDF-SS with restricted preemption on every configuration of Fig. 1, light and heavy load
    n = 96
    sp = W.CONFIGS[name](n).params
    algo = np.full(n, 4, np.uint8)
    cfg0 = (np.arange(n) % 12).astype(np.uint8)
    sim = B.MigSim(sp, n, seed)
    recs, tot = sim.alloc_recs(), sim.alloc_totals()
    sim.reset(0, dev(algo), dev(cfg0))
    sim.rollout(W.POLICY_STATIC, recs_out=recs, totals_out=tot)
    torch.cuda.synchronize()
    g_recs, g_tot = B.recs_to_numpy(recs), B.totals_to_numpy(tot)
    with cf.ProcessPoolExecutor(min(n, os.cpu_count() or 1)) as ex:
        res = list(ex.map(_oracle_static, [(sp, seed, e, 4, int(cfg0[e]), e < 12) for e in range(n)]))
    for e, o_recs, o_tot, o_trace in res:
        assert_same_records(g_recs[:, e], g_tot[e], o_recs, o_tot, "%s env %d cfg %d" % (name, e, cfg0[e]))
        if o_trace is not None:
            ev, t1 = sim.debug_trace(e, cap_events=400000)
            assert len(ev) == len(o_trace) and ev.tobytes() == o_trace.tobytes(), "env %d" % e
    sim.close()


@pytest.mark.parametrize("tile", [1, 16, 32])
def test_every_tile_width_gives_the_same_records(tile):
    for name, n in (("C2", 200), ("C3", 200)):
        wl = W.CONFIGS[name](n)
        _, recs_ref, tot_ref, _ = gpu_rollout(wl, sim=B.MigSim(wl.params, n, wl.seed, tile=8))
        sim = B.MigSim(wl.params, n, wl.seed, tile=tile)
        assert sim.get_tile() == tile
        _, recs, tot, _ = gpu_rollout(wl, sim=sim)
        assert tot.tobytes() == tot_ref.tobytes() and recs.tobytes() == recs_ref.tobytes()
        sim.close()


@pytest.mark.parametrize("entries", [0, 1, 7, 100])
def test_thread_kernel_arrival_lists_of_any_capacity_give_the_same_day(entries):
    # 0 = arrivals drawn inside the event loop; 1, 7, 100 = lists that fill up and are refilled many times a day
    for name, n in (("C3", 96), ("C4", 64)):
        wl = W.CONFIGS[name](n)
        _, recs_ref, tot_ref, _ = gpu_rollout(wl, sim=B.MigSim(wl.params, n, wl.seed, tile=1))
        sim = B.MigSim(wl.params, n, wl.seed, tile=1)
        sim.set_arrival_buffer(entries)
        _, recs, tot, _ = gpu_rollout(wl, sim=sim)
        assert tot.tobytes() == tot_ref.tobytes() and recs.tobytes() == recs_ref.tobytes()
        # step by step, switching the generator between epochs
        sim.reset(0, dev(wl.algo), dev(wl.cfg0))
        rec = torch.zeros((n, 64), dtype=torch.uint8, device="cuda")
        for k in range(24):
            sim.set_arrival_buffer(entries if k % 2 else (0 if entries else 50))
            sim.step(dev(recs_ref[k]["cfg"].astype(np.uint8)), rec_out=rec)
            torch.cuda.synchronize()
            assert B.recs_to_numpy(rec).tobytes() == recs_ref[k].tobytes(), (name, entries, k)
        sim.close()


@pytest.mark.parametrize("algo", [None, 4])
def test_c5_full_size_every_env_agrees_between_kernel_families(algo):
    # the two kernel families are independent implementations (warp tiles with an unordered table and argmin passes;
    # one thread per env with a sorted queue and pre-generated arrivals): every record and every trace hash of all
    # 65 536 env-days of BASELINE C5 must agree (the oracle checks a sample of the same days in test_c5_full_size_every_env)
    if B.DEFAULT_TILE != 1:
        pytest.skip("runs once")
    wl = W.CONFIGS["C5"](65536)
    if algo is not None:
        wl.algo[:] = algo                                     # EDF-SS with restricted preemption
    out = []
    for tile in (1, 8):
        sim, recs, tot, _ = gpu_rollout(wl, sim=B.MigSim(wl.params, 65536, wl.seed, tile=tile))
        out.append((recs, tot))
        sim.close()
    assert out[0][1].tobytes() == out[1][1].tobytes()
    assert out[0][0].tobytes() == out[1][0].tobytes()
    assert len(np.unique(out[0][1]["trace_hash"])) == 65536


@pytest.mark.parametrize("epw", [1, 4, 32])
def test_thread_kernel_envs_per_warp_gives_the_same_day(epw):
    for name, n in (("C3", 200), ("C4", 70)):
        wl = W.CONFIGS[name](n)
        _, recs_ref, tot_ref, _ = gpu_rollout(wl, sim=B.MigSim(wl.params, n, wl.seed, tile=8))
        sim = B.MigSim(wl.params, n, wl.seed, tile=1)
        sim.set_envs_per_warp(epw)
        _, recs, tot, _ = gpu_rollout(wl, sim=sim)
        assert tot.tobytes() == tot_ref.tobytes() and recs.tobytes() == recs_ref.tobytes()
        sim.close()
    with pytest.raises(B.MigError):
        sim = B.MigSim(wl.params, n, wl.seed, tile=1)
        sim.set_envs_per_warp(3)


def _random_setup(seed, n):
    """A random but valid parameter set: classes, speeds (not even monotone in the slice size), duration tables, slack
    ranges, a random subset of Fig. 1 plus a made-up partition, power tables, cap, rates, repartition costs, thresholds,
    a random bucket-dependent table, mixed algorithms."""
    rng = np.random.default_rng(1000 + seed)
    nc = int(rng.integers(1, 17))
    speeds = [[int(x) for x in rng.integers(1, 2000, size=5)] for _ in range(nc)]
    durs = []
    for _ in range(nc):
        q = np.sort(rng.integers(1, int(rng.choice([20, 200, 3000])), size=65))
        durs.append([int(x) for x in q])
    weights = [float(x) for x in rng.uniform(0.1, 1.0, size=nc)]
    cfgs = [W.FIG1_CONFIGS[i] for i in rng.choice(12, size=int(rng.integers(1, 12)), replace=False)]
    cfgs.append(((3, 0), (2, 3), (1, 5)))                               # not in Fig. 1: slot 6 unused
    sp = W.make_params(speeds, durs, weights, jobs_per_day=float(rng.choice([300, 2000, 9000])), amplitude=float(rng.uniform(0, 0.9)),
                       slack=(int(rng.integers(1024, 2000)), int(rng.integers(2000, 5000))), configs=tuple(cfgs),
                       cap=int(rng.choice([1, 5, 11, 12, 40, 256, 1024])), repart_downtime_s=int(rng.choice([0, 1, 4, 60, 900])),
                       repart_energy_mj=int(rng.choice([0, 1000, 6_000_000])), crit_laxity_s=int(rng.choice([0, 1, 60, 600])),
                       crit_max=int(rng.integers(0, 6)), job_limit=int(rng.choice([0, 0, 50])), decide_on_events=int(rng.integers(0, 2)))
    sp = dataclasses.replace(sp, curve_mw=rng.integers(0, 50000, size=8).astype(np.int32), p_idle_mw=rng.integers(0, 60000, size=5).astype(np.int32),
                             p_busy_mw=rng.integers(60000, 250000, size=5).astype(np.int32)).normalised()
    ncfg = len(cfgs)
    table = rng.integers(0, ncfg, size=(n, 24, 4)).astype(np.uint8)
    table[::5, :, :] = rng.integers(0, ncfg + 2, size=(len(table[::5]), 24, 4))    # some actions are invalid: stay + flag
    algo = rng.integers(0, 5, size=n).astype(np.uint8)
    cfg0 = rng.integers(0, ncfg, size=n).astype(np.uint8)
    return sp, table, algo, cfg0


@pytest.mark.parametrize("seed", range(10))
def test_random_parameter_sets(seed):
    # differential test over parameter space: both kernel families on every env, the oracle on a sample with full traces
    if B.DEFAULT_TILE != 1:
        pytest.skip("runs once")
    n = 48
    sp, table, algo, cfg0 = _random_setup(seed, n)
    out = []
    for tile in (1, 8):
        sim = B.MigSim(sp, n, 4242 + seed, tile=tile)
        recs, tot = sim.alloc_recs(), sim.alloc_totals()
        d_table = dev(table)
        sim.reset(seed, dev(algo), dev(cfg0))
        sim.rollout(W.POLICY_TABLE, table=d_table, recs_out=recs, totals_out=tot)
        torch.cuda.synchronize()
        out.append((B.recs_to_numpy(recs), B.totals_to_numpy(tot)))
        if tile == 1:
            traces = [sim.debug_trace(e, policy=W.POLICY_TABLE, table=d_table, cap_events=600000) for e in range(4)]
        sim.close()
    assert out[0][1].tobytes() == out[1][1].tobytes() and out[0][0].tobytes() == out[1][0].tobytes()
    for e in range(4):
        r = O.rollout(sp, 4242 + seed, e, episode=seed, algo=int(algo[e]), cfg0=int(cfg0[e]), policy=W.POLICY_TABLE, table=table[e], trace_cap=600000)
        assert_same_records(out[0][0][:, e], out[0][1][e], r.recs, r.totals, "seed %d env %d" % (seed, e))
        ev, t1 = traces[e]
        assert len(ev) == len(r.trace) and ev.tobytes() == r.trace.tobytes(), (seed, e)


def test_set_tile_between_kernel_families_needs_a_reset():
    wl = W.config_c3(32)
    sim = B.MigSim(wl.params, 32, wl.seed, tile=8)
    sim.reset(0, dev(wl.algo), dev(wl.cfg0))
    sim.set_tile(16)                                        # same saved-state layout: allowed mid-day
    sim.step(dev(wl.cfg0))
    sim.set_tile(1)                                         # another layout: the day must be restarted
    with pytest.raises(B.MigError) as ei:
        sim.step(dev(wl.cfg0))
    assert ei.value.code == B.MIG_ESTATE
    with pytest.raises(B.MigError):
        sim.set_tile(4)
    sim.close()


# ------------------------------------------------------------------------------------------------ Q-network
@pytest.mark.parametrize("B_", [1, 31, 32, 33, 1000, 8192])
def test_q_eval_bit_exact(B_):
    qw = W.make_qnet(7, 12)
    q = B.QNet(qw)
    rng = np.random.default_rng(B_)
    x = rng.uniform(0, 4, size=(B_, 64)).astype(np.float32)
    x[rng.uniform(size=x.shape) < 0.5] = 0.0
    q_out = torch.zeros((B_, 12), dtype=torch.float32, device="cuda")
    am = torch.zeros(B_, dtype=torch.uint8, device="cuda")
    q.q_eval(dev(x), q_out, am)
    torch.cuda.synchronize()
    ref_q, ref_am = O.q_eval(qw, x)
    assert q_out.cpu().numpy().tobytes() == ref_q.tobytes()
    assert np.array_equal(am.cpu().numpy(), ref_am)
    # and within north_star's 1e-4 relative of the float64 evaluation
    ref64 = O.q_eval_f64(qw, x)
    assert np.max(np.abs(q_out.cpu().numpy() - ref64) / np.maximum(np.abs(ref64), 1e-2)) < 1e-4


def test_q_eval_small_hidden_and_ties():
    qw = W.make_qnet(3, 5, hidden=64)
    qw.W3[:] = 0; qw.b3[:] = [1, 7, 7, 7, 0]
    q = B.QNet(qw)
    x = np.random.default_rng(0).normal(size=(40, 64)).astype(np.float32)
    am = torch.zeros(40, dtype=torch.uint8, device="cuda")
    q.q_eval(dev(x), None, am)
    assert np.all(am.cpu().numpy() == 1)


# ------------------------------------------------------------------------------------------------ edge cases
def test_queue_cap_overflows_shared_table_and_drops():
    sp = tiny_params(cap=256)
    rows = [(5, 0, 100, 100000)] * 300 + [(50000, 0, 7, 50100)] * 3
    ev, tot = gpu_script(sp, rows, 0, 3)
    r = O.rollout(sp, 0, 0, algo=0, cfg0=3, jobs=O.make_jobs(rows), trace_cap=4096)
    assert int(tot["n_dropped"]) == 44 and int(tot["n_sys_max"]) == 256
    assert ev.tobytes() == r.trace.tobytes() and tot.tobytes() == r.totals.tobytes()


@pytest.mark.parametrize("cap", [1, 3, 13])
def test_tiny_queue_caps(cap):
    # caps below the shared-memory ring / table sizes: admission, drops and every algorithm still agree with the oracle
    sp = tiny_params(speeds=(LINEAR, SUB05), cap=cap, crit_laxity_s=3)
    rng = np.random.default_rng(cap)
    rows = sorted((int(rng.integers(0, 400)), int(rng.integers(0, 2)), int(rng.integers(1, 30)), 0) for _ in range(120))
    rows = [(a, c, d, a + int(rng.integers(1, 200))) for (a, c, d, _) in rows]
    for algo in range(5):
        ev, tot = gpu_script(sp, rows, algo, 6, cap_events=4096)
        r = O.rollout(sp, 0, 0, algo=algo, cfg0=6, jobs=O.make_jobs(rows), trace_cap=4096)
        assert int(tot["n_dropped"]) > 0 and int(tot["n_sys_max"]) == cap
        assert ev.tobytes() == r.trace.tobytes() and tot.tobytes() == r.totals.tobytes(), (cap, algo)


@pytest.mark.parametrize("algo", [0, 1, 2, 3, 4])
def test_long_queue_all_algorithms(algo):
    # ~500 jobs in system (beyond the entries kept in shared memory), all 4 algorithms, mixed classes; the LLF / LALF
    # runs also raise several hundred critical-laxity events
    sp = tiny_params(speeds=(LINEAR, SUB05, CAP3), cap=1024, crit_laxity_s=30)
    rng = np.random.default_rng(algo)
    rows = sorted((int(rng.integers(0, 2000)), int(rng.integers(0, 3)), int(rng.integers(1, 30)), 0) for _ in range(700))
    rows = [(a, c, d, a + int(rng.integers(1, 4000))) for (a, c, d, _) in rows]
    ev, tot = gpu_script(sp, rows, algo, 5, cap_events=20000)
    r = O.rollout(sp, 0, 0, algo=algo, cfg0=5, jobs=O.make_jobs(rows), trace_cap=20000)
    assert int(tot["n_sys_max"]) > 200
    assert len(ev) == len(r.trace)
    assert ev.tobytes() == r.trace.tobytes() and tot.tobytes() == r.totals.tobytes()


def test_truncation_bad_action_and_empty_day():
    sp = tiny_params(t_limit_s=90000)
    ev, tot = gpu_script(sp, [(0, 0, 10, 50)], 0, 0)       # dur7 limited by the class table (10 s): finishes
    assert int(tot["status"]) == 0
    import dataclasses
    sp2 = dataclasses.replace(W.make_params([LINEAR], [W.dur_constant(100000)], [1], jobs_per_day=200, amplitude=0.0), t_limit_s=90000)
    ev, tot = gpu_script(sp2, [(0, 0, 100000, 50)], 0, 0)
    r = O.rollout(sp2, 0, 0, algo=0, cfg0=0, jobs=O.make_jobs([(0, 0, 100000, 50)]), trace_cap=100)
    assert int(tot["status"]) & 1 and tot.tobytes() == r.totals.tobytes() and ev.tobytes() == r.trace.tobytes()
    # bad action = stay + flag
    ev, tot = gpu_script(sp, [(10, 0, 5, 100)], 0, 3, actions=[200] * 24)
    assert int(tot["status"]) & 2 and int(tot["n_repart"]) == 0
    # a day with no arrivals at all (thinning threshold 0 ... only w_accept == 0 passes)
    sp3 = dataclasses.replace(W.config_c2(4).params, accept_thr=np.zeros(1440, np.uint32))
    sim = B.MigSim(sp3, 4, 1)
    tot = sim.alloc_totals()
    sim.reset(0, dev(np.arange(4, dtype=np.uint8)), dev(np.array([0, 3, 6, 11], np.uint8)))
    sim.rollout(W.POLICY_STATIC, totals_out=tot)
    t = B.totals_to_numpy(tot)
    assert np.all(t["n_jobs"] == 0) and np.all(t["n_events"] == 0) and np.all(t["t_end"] == 86400)
    for e, cfg in enumerate([0, 3, 6, 11]):
        idle = sum(int(sp3.p_idle_mw[W.SIZE_INDEX[int(g)]]) for g in sp3.size_at_slot[cfg] if g)
        assert int(t[e]["energy_mj"]) == idle * 86400
    sim.close()


def test_episode_changes_the_day_and_reset_is_repeatable():
    wl = W.config_c2(32)
    sim = B.MigSim(wl.params, 32, wl.seed)
    hashes = []
    for ep in (0, 1, 0):
        tot = sim.alloc_totals()
        sim.reset(ep, dev(wl.algo), dev(wl.cfg0))
        sim.rollout(W.POLICY_STATIC, totals_out=tot)
        hashes.append(B.totals_to_numpy(tot)["trace_hash"].copy())
    assert np.array_equal(hashes[0], hashes[2]) and not np.any(hashes[0] == hashes[1])
    r = O.rollout(wl.params, wl.seed, 5, episode=1, algo=int(wl.algo[5]), cfg0=int(wl.cfg0[5]))
    assert int(r.totals["trace_hash"]) == int(hashes[1][5])
    sim.close()
