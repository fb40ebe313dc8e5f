"""GPU parity of the extensions (readings #29-#32): the CUDA path (through the C ABI) vs the
oracle, bit for bit -- the MIG-disabled GPU as a configuration, the whole-GPU repartition penalty, the time per utilisation
level, the discounted return, the BINNED policy (hourly and event-driven), the paper's benchmark policies (No-MIG, static
configuration 3, day / night), the ET reduction.  Every test runs on both kernel families: one thread per environment (the
library default) and warp tiles of 8, 16 and 32 lanes per environment (mig_sim_set_tile).
"""
import dataclasses

import numpy as np
import pytest
import torch

import trace_check
from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
from util import LINEAR, SUB05, golden, tiny_params

pytestmark = pytest.mark.gpu

G = golden("handworked_ext.json")
G1 = golden("handworked.json")
B = None


@pytest.fixture(scope="module", autouse=True, params=[1, 8, 16, 32], ids=["thread", "tile8", "tile16", "tile32"])
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


def gpu_day(sp, n, seed, algo, cfg0, policy=0, table=None, jobs=None, want_util=False):
    """One rollout of n envs; returns records, totals, discounted returns, utilisation levels (or None), the handle."""
    sim = B.MigSim(sp, n, seed)
    if jobs is not None:
        sim.debug_set_jobs(jobs)
    recs, tot = sim.alloc_recs(), sim.alloc_totals()
    sim.reset(0, dev(np.asarray(algo, np.uint8)), dev(np.asarray(cfg0, np.uint8)))
    d_table = None if table is None else dev(table)
    sim.rollout(policy, table=d_table, recs_out=recs, totals_out=tot)
    ret = torch.zeros(n, dtype=torch.float32, device="cuda")
    util = torch.zeros((n, 8), dtype=torch.int32, device="cuda") if want_util else None
    sim.aux(return_out=ret, util_s_out=util)
    torch.cuda.synchronize()
    return B.recs_to_numpy(recs), B.totals_to_numpy(tot), ret.cpu().numpy(), None if util is None else util.cpu().numpy(), sim, d_table


def compare_days(sp, n, seed, algo, cfg0, policy=0, table=None, per_env_table=True, trace_envs=(0,), jobs=None):
    want_util = bool(sp.util_hist)
    recs, tot, ret, util, sim, d_table = gpu_day(sp, n, seed, algo, cfg0, policy, table, jobs, want_util)
    ph = O.ParamsHolder(sp)
    for e in range(n):
        tb = None if table is None else (table[e] if per_env_table else table)
        r = O.rollout(ph, seed, e, algo=int(algo[e]), cfg0=int(cfg0[e]), policy=policy, table=tb, jobs=jobs,
                      trace_cap=400000 if e in trace_envs else 0)
        assert tot[e].tobytes() == r.totals.tobytes(), (e, tot[e], r.totals)
        assert recs[:, e].tobytes() == r.recs.tobytes(), e
        assert np.float32(ret[e]).tobytes() == np.float32(r.ret).tobytes(), (e, ret[e], r.ret)
        if want_util:
            assert util[e].tolist() == r.util.tolist(), (e, util[e], r.util)
        if e in trace_envs:
            ev, t1 = sim.debug_trace(e, policy=policy, table=d_table)
            assert len(ev) == len(r.trace), (e, len(ev), len(r.trace))
            if ev.tobytes() != r.trace.tobytes():
                i = int(np.nonzero(ev != r.trace)[0][0])
                raise AssertionError("env %d: first differing event %d:\n gpu %s\n orc %s" % (e, i, ev[max(0, i - 3):i + 2], r.trace[max(0, i - 3):i + 2]))
            assert t1.tobytes() == r.totals.tobytes()
    sim.close()
    return recs, tot


# ------------------------------------------------------------------------------------------------ hand-worked, direct
def test_handworked_N_O_Q_direct_on_the_gpu():
    # the expected values of the golden file, checked against the CUDA path itself (not through the oracle)
    g = G["N"]
    cfgs = tuple(tuple((s, p) for s, p in row) for row in g["configs"])
    sp = dataclasses.replace(tiny_params(speeds=(LINEAR, SUB05), configs=cfgs), speed_nomig=np.array(g["speed_nomig"], np.uint32),
                             p_idle_nomig_mw=g["p_idle_nomig_mw"], p_busy_nomig_mw=g["p_busy_nomig_mw"], util_hist=1)
    jobs = np.array([tuple(j) for j in g["jobs"]], dtype=B.JOB_DTYPE)
    recs, tot, ret, util, sim, _ = gpu_day(sp, 1, 0, [g["algo"]], [0], jobs=jobs, want_util=True)
    assert int(recs[0, 0]["energy_mj"]) == g["epoch0_energy_mj"] and int(tot[0]["energy_mj"]) == g["day_energy_mj"]
    assert int(tot[0]["busy_unit_s"]) == g["busy_unit_s"] and util[0].tolist() == g["util"] and int(tot[0]["tardiness_s"]) == g["tardiness"]
    ev, _ = sim.debug_trace(0)
    assert {int(e["job"]): int(e["t"]) for e in ev if e["type"] == 5} == {int(k): v for k, v in g["completion_nomig"].items()}
    sim.close()
    # O: whole GPU down
    d, o = G1["D"], G["O"]
    sp = dataclasses.replace(tiny_params(repart_downtime_s=d["downtime_s"], repart_energy_mj=d["repart_energy_mj"]), repart_all_down=1, util_hist=1)
    table = np.full((1, 24, 4), d["action_epoch1"], dtype=np.uint8); table[0, 0, :] = d["cfg0"]
    jobs = np.array([tuple(j) for j in d["jobs"]], dtype=B.JOB_DTYPE)
    recs, tot, ret, util, sim, _ = gpu_day(sp, 1, 0, [d["algo"]], [d["cfg0"]], policy=W.POLICY_TABLE, table=table, jobs=jobs, want_util=True)
    assert int(recs[1, 0]["energy_mj"]) == o["epoch1_energy_mj"] and int(recs[1, 0]["n_preempt"]) == o["epoch1_n_preempt"]
    assert util[0].tolist() == G["P"]["util_O"]
    sim.close()
    # Q: discounted return
    q = G["Q"]
    sp = dataclasses.replace(tiny_params(day_s=q["n_epochs"] * 3600, n_epochs=q["n_epochs"], w_energy=q["w_energy"], w_tardy=q["w_tardy"]), gamma=q["gamma"])
    jobs = np.array([tuple(j) for j in q["jobs"]], dtype=B.JOB_DTYPE)
    recs, tot, ret, util, sim, _ = gpu_day(sp, 1, 0, [0], [0], jobs=jobs)
    assert float(ret[0]) == q["return"]
    sim.close()


# ------------------------------------------------------------------------------------------------ generated days
@pytest.mark.parametrize("kind", ["nomig", "static", "daynight"])
def test_paper_benchmark_policies(kind):
    # full GPU without MIG, static configuration 3, day / night 6 <-> 2; whole-GPU 4 s penalty, discounted
    # return, utilisation levels; every algorithm (the paper runs restricted-preemption EDF-SS)
    n = 40
    wl = W.config_benchmark(kind, n)
    algo = (np.arange(n) % 5).astype(np.uint8)
    compare_days(wl.params, n, wl.seed, algo, wl.cfg0, wl.policy, wl.table, trace_envs=(0, 1, 2, 3, 4))


def test_mig_disabled_among_random_repartitions():
    # hourly random actions over all 13 configurations (12 of Fig. 1 + MIG disabled), whole-GPU penalty on and off
    n = 30
    for all_down in (0, 1):
        sp = dataclasses.replace(W.benchmark_params(repart_downtime_s=7, repart_energy_mj=1_000_000), repart_all_down=all_down)
        rng = np.random.default_rng(50 + all_down)
        table = np.repeat(rng.integers(0, 13, size=(n, 24, 1)).astype(np.uint8), 4, axis=2)
        compare_days(sp, n, 21, (np.arange(n) % 5).astype(np.uint8), rng.integers(0, 13, size=n).astype(np.uint8), W.POLICY_TABLE, table,
                     trace_envs=(0, 1, 2, 3, 4))


@pytest.mark.parametrize("rate,split", [("0.1", "80"), ("0.75", "80"), ("0.5", "20")])
def test_sweep_parameter_sets(rate, split):
    # Figs. 7-10 are parameter files: arrival rate 0.1 / 0.75 (x0.2 / x1.5 of the default), 20 % inference split
    n = 20
    sp = W.benchmark_params(jobs_per_day=2000.0 * W.SWEEP_RATE_SCALE[rate], inference_frac=W.SWEEP_INFERENCE[split])
    compare_days(sp, n, 31, (np.arange(n) % 4).astype(np.uint8), (np.arange(n) % 12).astype(np.uint8), trace_envs=(0,))


# ------------------------------------------------------------------------------------------------ BINNED policy
def _random_binned_table(sp, rng, p_stay=0.7):
    Bc = sp.binned_codes
    t = rng.integers(0, sp.n_configs, size=(sp.n_configs, sp.n_tbins, Bc, Bc, Bc)).astype(np.uint8)
    stay = rng.random(t.shape) < p_stay
    for c in range(sp.n_configs):
        t[c][stay[c]] = c
    return t


@pytest.mark.parametrize("event_driven", [0, 1])
def test_binned_policy_random_tables(event_driven):
    # a random table over the binned 2+2m state, consulted hourly or after every arrival / completion
    n = 30
    sp = W.binned_defaults(dataclasses.replace(W.benchmark_params(jobs_per_day=800.0, repart_downtime_s=4), decide_on_events=event_driven))
    rng = np.random.default_rng(60 + event_driven)
    table = _random_binned_table(sp, rng, 0.97 if event_driven else 0.5)
    recs, tot = compare_days(sp, n, 41, (np.arange(n) % 5).astype(np.uint8), (np.arange(n) % 13).astype(np.uint8), W.POLICY_BINNED, table,
                             per_env_table=False, trace_envs=(0, 1, 2, 3, 4, 5))
    assert int(tot["n_repart"].sum()) > n                     # the table does move the configuration


def test_binned_policy_handworked_J():
    j = G1["J"]
    sp = dataclasses.replace(tiny_params(repart_downtime_s=j["downtime_s"], repart_energy_mj=j["repart_energy_mj"]), decide_on_events=1,
                             n_tbins=24, dbin_edges=np.array([0, 3600], np.int32), abin_edges=np.array([8000, 20000], np.int32))
    Bc = sp.binned_codes
    t = np.zeros((sp.n_configs, 24, Bc, Bc, Bc), dtype=np.uint8)
    t[:, :, 0] = j["table"]["bucket0"]; t[:, :, 1:] = j["table"]["bucket1_3"]
    jobs = np.array([tuple(x) for x in j["jobs"]], dtype=B.JOB_DTYPE)
    recs, tot, ret, util, sim, d_table = gpu_day(sp, 1, 0, [j["algo"]], [j["cfg0"]], policy=W.POLICY_BINNED, table=t, jobs=jobs)
    ev, _ = sim.debug_trace(0, policy=W.POLICY_BINNED, table=d_table)
    names = {1: "ARRIVE", 2: "DROP", 3: "START", 4: "PREEMPT", 5: "COMPLETE", 6: "CRIT", 7: "SLICE_UP", 8: "REPART"}
    assert [[int(e["t"]), names[int(e["type"])], int(e["job"]), int(e["slot"])] for e in ev] == j["events"]
    assert int(recs[0, 0]["energy_mj"]) == j["epoch0_energy_mj"]
    sim.close()


# ------------------------------------------------------------------------------------------------ step API, boundary
def test_step_api_keeps_return_and_levels():
    # 24 mig_sim_step calls with the day / night actions = the rollout (records, return, utilisation levels)
    n = 16
    wl = W.config_benchmark("daynight", n)
    recs_r, tot_r, ret_r, util_r, sim, _ = gpu_day(wl.params, n, wl.seed, wl.algo, wl.cfg0, wl.policy, wl.table, want_util=True)
    sim.close()
    sim = B.MigSim(wl.params, n, wl.seed)
    sim.reset(0, dev(wl.algo), dev(wl.cfg0))
    rew = torch.zeros(n, dtype=torch.float32, device="cuda")
    G_ = np.zeros(n, dtype=np.float32); disc = np.float32(1.0)
    for k in range(24):
        sim.step(dev(wl.table[:, k, 0].copy()), reward_out=rew)
    tot = sim.alloc_totals(); sim.totals(tot)
    ret = torch.zeros(n, dtype=torch.float32, device="cuda"); util = torch.zeros((n, 8), dtype=torch.int32, device="cuda")
    sim.aux(return_out=ret, util_s_out=util)
    torch.cuda.synchronize()
    assert B.totals_to_numpy(tot).tobytes() == tot_r.tobytes()
    assert ret.cpu().numpy().tobytes() == ret_r.tobytes() and util.cpu().numpy().tobytes() == util_r.tobytes()
    sim.close()


def test_boundary_errors_of_the_extensions():
    sp = W.benchmark_params()
    sim = B.MigSim(sp, 4, 1)
    assert sim.get_tile() == B.DEFAULT_TILE
    with pytest.raises(B.MigError):
        sim.rollout(W.POLICY_BINNED, table=dev(np.zeros(16, np.uint8)))      # (reset not called / no bins)
    sim.close()
    bad = dataclasses.replace(sp, speed_nomig=None)           # size code 8 without its speed column
    with pytest.raises(B.MigError) as ei:
        B.MigSim(bad, 4, 1)
    assert ei.value.code == B.MIG_EINVAL
    cfgs = W.FIG1_CONFIGS + (((8, 0), (1, 6)),)              # the MIG-disabled GPU is not alone
    bad = dataclasses.replace(sp, size_at_slot=W.size_at_slot_table(cfgs))
    with pytest.raises(B.MigError):
        B.MigSim(bad, 4, 1)
    plain = tiny_params()
    sim = B.MigSim(plain, 4, 1)
    sim.reset(0, dev(np.zeros(4, np.uint8)), dev(np.zeros(4, np.uint8)))
    with pytest.raises(B.MigError) as ei:
        sim.aux(util_s_out=torch.zeros((4, 8), dtype=torch.int32, device="cuda"))     # util_hist was off
    assert ei.value.code == B.MIG_ESTATE
    sim.close()


def test_et_reduce_matches_the_oracle_and_the_hand_values():
    g = G["T"]
    et, a = B.et_reduce(g["x"], g["y"], g["group"], 2)
    assert abs(a - g["a"]) < 1e-15 and all(abs(et[k] - g["et_num"][k] / g["et_den"]) < 1e-12 for k in range(2))
    # ET of the paper's three benchmark policies from simulated days (energy, average tardiness per simulation)
    xs, ys, gs = [], [], []
    for gi, kind in enumerate(("nomig", "static", "daynight")):
        wl = W.config_benchmark(kind, 24)
        recs, tot, ret, util, sim, _ = gpu_day(wl.params, 24, wl.seed, wl.algo, wl.cfg0, wl.policy, wl.table)
        sim.close()
        xs += [float(v) for v in tot["energy_mj"]]
        ys += [float(t) / max(1, int(c)) for t, c in zip(tot["tardiness_s"], tot["n_completed"])]
        gs += [gi] * 24
    et, a = B.et_reduce(xs, ys, gs, 3)
    eo, ao = O.et_reduce(xs, ys, gs, 3)
    assert np.allclose(et, eo, rtol=1e-13, atol=0) and abs(a - ao) <= 1e-13 * ao
    assert et[2] < et[1] < et[0]        # day/night < static cfg 3 < No-MIG on this workload, the order of the paper's Table III
