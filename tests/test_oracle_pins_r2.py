"""Pins for the four parts of the oracle that round 1 left unpinned ("What's weak" #1):

  (a) orc_env_observe -- all 64 entries of the state vector at three hand-worked snapshots (golden K);
  (b) the duration draw of gen_next -- distribution against the table's own law + the bit fields of reading R5;
  (c) the curve_mw[U] term of power_now -- hand-worked B and D re-run with a non-zero curve (golden L);
  (d) the load-bucket borders 1 / 8 / 64 of the tabulated policy (golden M).

Expected values are in tests/golden/handworked_r2.json with the arithmetic beside them; none was produced by running an
implementation.  Each test was checked to FAIL under a one-line mutation of oracle/mig_oracle.c (listed per test).
"""
import dataclasses
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
from util import LINEAR, SUB05, golden, tiny_params

G1 = golden("handworked.json")
G2 = golden("handworked_r2.json")


def _dense(d):
    x = np.zeros(64, dtype=np.float32)
    for k, v in d.items():
        x[int(k)] = v
    return x


# ------------------------------------------------------------------------------------------------ (a) state vector
def test_K_state_vector_all_64_entries():
    # mutations that fail here: x[16+q] = 1.0 for a down slice; size/7 instead of /8; (t/3600+1)%24; n_wait/32;
    # first-3 in id order (J0 would come first); due order without the id tie rule (x[60], x[61] swap);
    # rd_fastest_cfg instead of rd_mean_cfg; mean over UP slices only (J3: 6550); missing clamp at 32767; missing
    # clamp at 0 of overdue deadlines (none: it must be NEGATIVE); last_epoch_drops from the totals instead of the epoch
    g = G2["K"]
    sp = tiny_params(speeds=(LINEAR, SUB05), cap=g["cap"], repart_downtime_s=g["downtime_s"], repart_energy_mj=g["repart_energy_mj"])
    env = O.Env(sp, 0, 0, jobs=O.make_jobs(g["jobs"]), trace_cap=256)
    x0 = env.reset(algo=g["algo"], cfg0=g["cfg0"])
    assert np.array_equal(x0, _dense(g["state_0"])), np.nonzero(x0 != _dense(g["state_0"]))
    x1, _, _, _, rec = env.step(g["actions"][0])
    assert np.array_equal(x1, _dense(g["state_3600"])), (np.nonzero(x1 != _dense(g["state_3600"])), x1)
    assert int(rec[0]["n_dropped"]) == 0
    x2, _, _, _, rec = env.step(g["actions"][1])
    assert np.array_equal(x2, _dense(g["state_7200"])), (np.nonzero(x2 != _dense(g["state_7200"])), x2)
    assert int(rec[0]["n_dropped"]) == 2 and int(rec[0]["n_sys_end"]) == 5 and int(rec[0]["tardiness_s"]) == 33
    # the entries are the fractions written in the golden file's arithmetic (binary fractions: exact in fp32 and in JSON)
    assert x1[59] == np.float32(10577 / 4096) and x1[60] == np.float32(32767 / 4096)
    assert x2[56] == np.float32(-1200 / 4096) and x2[59] == np.float32(7642 / 4096) and x2[61] == np.float32(8167 / 4096)


def test_state_vector_slot_cover_and_hole():
    # cfg 5 {3g@0, 3g@4}: slot 3 is a hole and stays 0 in both the occupancy and the size rows
    sp = tiny_params()
    env = O.Env(sp, 0, 0, jobs=O.make_jobs([(10, 0, 10000, 50000)]))
    env.reset(algo=0, cfg0=4)
    x, *_ = env.step(4)
    want = np.zeros(64, np.float32)
    want[16:19] = 1.0                       # J0 on 3g@0 (ties -> lower slot), 3g@4 free, slot 3 a hole
    want[23] = 3 / 8; want[27] = 3 / 8
    want[31] = 1.0; want[55] = 1 / 8; want[63] = 1.0
    want[56] = 32767 / 4096                 # due - t = 46400 clamps to 32767
    want[59] = 19744 / 4096                 # rem = 8400000 - 3590*360 = 7107600; ceil(/360) = 19744 on both slices
    assert np.array_equal(x, want), np.nonzero(x != want)


# ------------------------------------------------------------------------------------------------ (b) duration draw
def _arrival_dur7(sp, seed, n_env, env0=0):
    """dur7 of every job of the generated days, read off the trace: with the slack multiplier fixed at 1.0 (Q10 1024) an
    ARRIVE / DROP event carries due = tick + dur7 (R5), whatever the scheduler does with the job afterwards."""
    assert np.all(sp.slack_q10 == 1024)
    out = {}
    for e in range(env0, env0 + n_env):
        r = O.rollout(sp, seed, e, algo=0, cfg0=0, trace_cap=200000)
        tr = r.trace[(r.trace["type"] == O.EV_ARRIVE) | (r.trace["type"] == O.EV_DROP)]
        assert len(tr) == int(r.totals["n_jobs"])
        out[e] = (tr["job"].astype(np.int64), tr["value"].astype(np.int64) - tr["t"].astype(np.int64))
    return out


def test_duration_draw_is_the_tables_distribution():
    # dur_uniform(100, 6500): q[i] = 100 + 100 i, so R5's draw q[i] + ((q[i+1] - q[i]) f >> 10) covers the integers
    # 100..6499 evenly.  Mutations that fail here: no interpolation (only multiples of 100 appear); i = w >> 27 (half of
    # the table); f >> 11 (the upper half of every segment is never drawn); q[i+1] + ... (shifted mean)
    sp = W.make_params([LINEAR], [W.dur_uniform(100, 6500)], [1], jobs_per_day=400, amplitude=0.0, cap=1024, slack=(1024, 1024),
                       t_limit_s=90000)
    assert list(sp.dur7_q[0][:3]) == [100, 200, 300] and int(sp.dur7_q[0][64]) == 6500
    d = np.concatenate([v[1] for v in _arrival_dur7(sp, 77, 100).values()])
    n = d.size
    assert n > 38000
    assert d.min() >= 100 and d.max() <= 6499 and d.min() < 110 and d.max() > 6490
    sd = 6400 / math.sqrt(12)
    assert abs(d.mean() - 3299.5) < 4.5 * sd / math.sqrt(n)
    assert abs(d.var() / (6400 ** 2 / 12) - 1.0) < 4.5 * math.sqrt(0.8 / n)          # uniform: var of s^2 = (kurt-1)/n sigma^4, kurt = 1.8
    # Kolmogorov-Smirnov against U[100, 6500)
    xs = np.sort(d)
    cdf = (xs - 100 + 1) / 6400.0
    ks = max(np.max(np.abs(cdf - np.arange(1, n + 1) / n)), np.max(np.abs((xs - 100) / 6400.0 - np.arange(0, n) / n)))
    assert ks < 1.95 / math.sqrt(n), ks                                             # P < 1e-3; a 64-step staircase has D = 1/64 = 0.0156
    # inside a segment every offset 0..99 is drawn: chi-square of dur7 mod 100 (99 dof) against the law of
    # floor(100 f / 1024), f uniform on 0..1023 (each offset has 10 or 11 of the 1024 values of f)
    p_off = np.bincount((100 * np.arange(1024)) >> 10, minlength=100) / 1024.0
    h = np.bincount(d % 100, minlength=100)
    chi2 = float(((h - n * p_off) ** 2 / (n * p_off)).sum())
    assert chi2 < 160.0, chi2                                                        # P(chi2_99 > 160) ~ 1e-4
    # segments are equally likely: chi-square of the segment index (63 dof)
    h = np.bincount((d - 100) // 100, minlength=64)
    chi2 = float(((h - n / 64.0) ** 2 / (n / 64.0)).sum())
    assert chi2 < 115.0, chi2


def test_duration_draw_bit_fields_of_reading_R5():
    # Which bits of w_dur select the segment and the offset is a READING (R5: i = w >> 26, f = (w >> 16) & 0x3FF),
    # not something the distribution can tell.  A table whose segment slopes are all different makes dur7 identify (i, f):
    # q[i] = 500 i^2 + 1, so dur7 - q[i] = ((1000 i + 500) f) >> 10.  w_dur comes from the Philox that
    # test_oracle_generator.py pins against ATen's engine: counter (k, stream 1, env, episode).
    q = [500 * i * i + 1 for i in range(65)]
    sp = W.make_params([LINEAR], [q], [1], jobs_per_day=3000, amplitude=0.0, cap=1024, slack=(1024, 1024), t_limit_s=90000)
    seed, env_id = 0x1234567811223344, 5
    # homogeneous arrivals: every candidate is accepted (thr = 2^32 - 1), so job id == candidate index k
    assert np.all(sp.accept_thr == 0xFFFFFFFF)
    ids, dur = _arrival_dur7(sp, seed, 1, env0=env_id)[env_id]
    assert len(ids) > 2500 and np.array_equal(ids, np.arange(len(ids)))
    seen_i = set()
    for k in range(2000):
        w = int(O.philox(k, 1, env_id, 0, seed & 0xFFFFFFFF, seed >> 32)[0])
        i, f = w >> 26, (w >> 16) & 0x3FF
        seen_i.add(i)
        assert int(dur[k]) == q[i] + (((q[i + 1] - q[i]) * f) >> 10), (k, hex(w), int(dur[k]))
    assert len(seen_i) == 64
    # two words by hand: w = 0xFFFF0000 -> i = 63, f = 1023: 1984501 + (63500*1023 >> 10) = 1984501 + 63437;
    #                    w = 0x04010000 -> i = 1,  f = 1:    501 + (1500 >> 10) = 502
    assert q[63] + ((63500 * 1023) >> 10) == 2047938 and q[1] + (1500 >> 10) == 502


# ------------------------------------------------------------------------------------------------ (c) curve_mw term
def _with_curve(sp):
    return dataclasses.replace(sp, curve_mw=np.array(G2["L"]["curve_mw"], dtype=np.int32)).normalised()


@pytest.mark.parametrize("name,algo", [("EDF-FS", 0), ("EDF-SS", 1)])
def test_L_curve_term_on_handworked_B(name, algo):
    # mutations that fail here: curve_mw[number of busy SLICES]; curve added only while U > 0; curve_mw[u] omitted
    g = G1["B"]
    r = O.rollout(_with_curve(tiny_params()), 0, 0, algo=algo, cfg0=g["cfg"], jobs=O.make_jobs(g["jobs"]), trace_cap=64)
    assert int(r.recs[0]["energy_mj"]) == G2["L"]["B"][name]["epoch0_energy_mj"]
    assert int(r.recs[1]["energy_mj"]) == (g["idle_mw"] + 500) * 3600            # idle config: curve_mw[0] all hour


def test_L_curve_term_on_handworked_D_repartition():
    g = G1["D"]
    sp = _with_curve(tiny_params(repart_downtime_s=g["downtime_s"], repart_energy_mj=g["repart_energy_mj"]))
    env = O.Env(sp, 0, 0, jobs=O.make_jobs(g["jobs"]))
    env.reset(algo=g["algo"], cfg0=g["cfg0"])
    _, _, dE0, _, _ = env.step(g["cfg0"])
    _, _, dE1, _, _ = env.step(g["action_epoch1"])
    assert dE0 == G2["L"]["D"]["epoch0_energy_mj"]
    assert dE1 == G2["L"]["D"]["epoch1_energy_mj"]


# ------------------------------------------------------------------------------------------------ (d) bucket borders
def _M_jobs():
    rows = []
    for t, n in G2["M"]["jobs_spec"]:
        rows += [(t, 0, 20000, t + 40000)] * n
    return rows


@pytest.mark.parametrize("event_driven", [0, 1])
def test_M_load_bucket_borders(event_driven):
    # mutations that fail here: n <= 8 / n < 9 / n < 7 (epoch 3 or 2 picks another column); n < 63 / n <= 64 (epoch 4 or 5);
    # n <= 0 ... n < 1 variants (epoch 1); bucket from n_wait instead of n_sys (epoch 2: 6 waiting + 1 running on cfg 6)
    g = G2["M"]
    table = np.full((24, 4), g["rest_of_day_cfg"], dtype=np.uint8)
    table[:6] = np.array(g["table_rows"], dtype=np.uint8)
    assert [g["table_rows"][k][g["bucket"][k]] for k in range(6)] == g["cfg_of_epoch"]
    sp = dataclasses.replace(tiny_params(cap=256), decide_on_events=event_driven)
    rows = _M_jobs()
    r = O.rollout(sp, 0, 0, algo=g["algo"], cfg0=g["cfg0"], policy=W.POLICY_TABLE, table=table, jobs=O.make_jobs(rows), trace_cap=4096)
    assert [int(c) for c in r.actions[:6]] == g["cfg_of_epoch"]
    if not event_driven:
        assert [int(c) for c in r.recs["cfg"][:6]] == g["cfg_of_epoch"]
        assert [0] + [int(n) for n in r.recs["n_sys_end"][:5]] == g["n_sys_at_epoch_start"]
    else:
        # reading #27: the row of the running epoch is looked up again after each tick with an arrival.  Epoch 1: 6 arrivals
        # at 3700 -> n_sys = 7 -> still column 1; epoch 2: the arrival at 7300 makes n_sys = 8 -> column 2 (cfg 10);
        # epoch 4: the arrival at 14500 makes n_sys = 64 -> column 3 (cfg 8)
        reparts = [(int(ev["t"]), int(ev["aux"]) & 0xFF) for ev in r.trace if ev["type"] == O.EV_REPART]
        assert reparts[:8] == [(100, 1), (3600, 5), (7200, 9), (7300, 10), (10800, 3), (14400, 7), (14500, 8), (18000, 0)], reparts
    assert int(r.totals["status"]) == 0 and int(r.totals["n_completed"]) == 64
