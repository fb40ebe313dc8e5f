"""Pins the oracle's random-draw path (readings R1-R7): Philox4x32-10, the integer -log2, the
thinning generator and the job attributes -- against things other than itself:

* Philox words vs PyTorch's header-only at::Philox4_32 (an independent implementation shipped with the wheel),
  compiled from tests/golden/philox_aten_ref.cpp;  structural properties of the bijection;
* the fixed-point -log2 vs double precision math.log2;
* Poisson statistics (mean = variance = N, hourly histogram proportional to the integrated rate), class
  frequencies, slack range;  M/D/1 mean wait (Pollaczek-Khinchine closed form).
"""
import math
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W
from util import GOLDEN, LINEAR


# ----------------------------------------------------------------------------------------------- Philox
@pytest.fixture(scope="module")
def aten_philox(tmp_path_factory):
    import torch.utils.cpp_extension as ce
    exe = str(tmp_path_factory.mktemp("philox") / "philox_aten_ref")
    inc = []
    for p in ce.include_paths():
        inc += ["-I", p]
    subprocess.run(["g++", "-O1", "-std=c++17", *inc, os.path.join(GOLDEN, "philox_aten_ref.cpp"), "-o", exe], check=True)

    def call(rows):
        text = "".join("%x %x %x %x %x %x\n" % tuple(r) for r in rows)
        out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout.split("\n")
        return [tuple(int(x, 16) for x in line.split()) for line in out if line.strip()]
    return call


def test_philox_matches_aten_engine(aten_philox):
    rng = np.random.default_rng(7)
    rows = [(0, 0, 0, 0, 0, 0), (0xFFFFFFFF,) * 6, (1, 0, 0, 0, 0, 0), (0, 1, 0, 0, 0, 0), (0, 0, 1, 0, 0, 0),
            (0, 0, 0, 1, 0, 0), (0, 0, 0, 0, 1, 0), (0, 0, 0, 0, 0, 1)]
    rows += [tuple(int(x) for x in rng.integers(0, 2 ** 32, size=6)) for _ in range(200)]
    # the layout the simulator uses: counter = (index, stream, env, episode), key = seed
    rows += [(k, s, e, ep, 3, 0) for k in (0, 1, 31, 32, 4095) for s in (0, 1, 2) for e in (0, 1, 65535) for ep in (0, 5)]
    ref = aten_philox(rows)
    assert len(ref) == len(rows)
    for r, w in zip(rows, ref):
        assert tuple(int(x) for x in O.philox(*r)) == w, r


def test_philox_counter_sensitivity():
    # a bijection of the counter for a fixed key: distinct counters -> distinct blocks; every word changes
    base = O.philox(5, 0, 9, 0, 11, 13)
    seen = {tuple(base)}
    for pos in range(4):
        c = [5, 0, 9, 0]
        c[pos] += 1
        w = O.philox(*c, 11, 13)
        assert tuple(w) not in seen
        seen.add(tuple(w))
        assert all(int(a) != int(b) for a, b in zip(w, base))
    words = np.array([O.philox(k, 0, 0, 0, 1, 0) for k in range(4096)], dtype=np.uint64)
    # uniformity: mean of 16384 words / 2^32 within 4 sigma of 0.5
    u = words.reshape(-1) / 4294967296.0
    assert abs(u.mean() - 0.5) < 4 * (1 / math.sqrt(12)) / math.sqrt(u.size)
    bits = ((words.reshape(-1)[:, None] >> np.arange(32, dtype=np.uint64)) & 1).mean(axis=0)
    assert np.all(np.abs(bits - 0.5) < 0.02)


# ----------------------------------------------------------------------------------------------- -log2
def test_log_table_definition():
    T = O.log_table()
    assert T[0] == 0 and T[256] == 1 << 24
    assert np.all(np.diff(T.astype(np.int64)) > 0) and np.all(np.diff(T.astype(np.int64)) < (1 << 17))
    for i in (1, 2, 17, 128, 255):
        assert abs(int(T[i]) - (2 ** 24) * math.log2(1 + i / 256.0)) <= 0.5


def test_neglog2_against_double():
    rng = np.random.default_rng(3)
    ws = [0, 1, 2, 3, 0x7FFFFFFF, 0x80000000, 0x80000001, 0xFFFFFFFF, 0xFFFFFFFE, 0x00010000, 0x00FFFFFF]
    ws += [int(x) for x in rng.integers(0, 2 ** 32, size=4000)]
    ws += [int(x) for x in rng.integers(0, 2 ** 12, size=200)]
    for w in ws:
        e24 = O.neglog2_q24(w)
        exact = -math.log2((w | 1) / 4294967296.0)
        # linear interpolation on 256 intervals: max error (1/8)(1/256)^2 log2(e) ~ 2.8e-6 bits, + quantisation
        assert abs(e24 / 16777216.0 - exact) < 4e-6, hex(w)
        assert 0 <= e24 <= 32 << 24


def test_neglog2_monotone():
    prev = None
    for w in range(1, 1 << 16, 2):
        v = O.neglog2_q24(w << 16)
        if prev is not None:
            assert v <= prev
        prev = v


# ----------------------------------------------------------------------------------------------- arrivals
def _arrivals(sp, seed, env, episode=0):
    r = O.rollout(sp, seed, env, episode=episode, algo=0, cfg0=0, trace_cap=20000)
    arr = r.trace[(r.trace["type"] == 1) | (r.trace["type"] == 2)]
    return r, arr


def _light_params(n_per_day, amplitude, n_classes=1, **kw):
    # 1 s jobs on a single 7g slice: queueing is irrelevant, only the generator matters
    speeds = [LINEAR] * n_classes
    durs = [W.dur_uniform(1, 3)] * n_classes
    return W.make_params(speeds, durs, kw.pop("weights", [1] * n_classes), jobs_per_day=n_per_day, amplitude=amplitude, **kw)


def test_poisson_count_mean_equals_variance():
    sp = _light_params(300, 0.0)
    counts = np.array([int(_arrivals(sp, 11, e)[0].totals["n_jobs"]) for e in range(600)], dtype=np.float64)
    n = counts.size
    # Poisson(300): sd of the mean = sqrt(300/n); sd of the sample variance ~ 300*sqrt(2/(n-1)) (+ small kurtosis term)
    assert abs(counts.mean() - 300.0) < 4 * math.sqrt(300.0 / n)
    assert abs(counts.var(ddof=1) - 300.0) < 4.5 * 300.0 * math.sqrt(2.0 / (n - 1))


def test_diurnal_histogram_follows_rate():
    A = 0.6
    sp = _light_params(1000, A)
    hist = np.zeros(24)
    tot = 0
    for e in range(120):
        _, arr = _arrivals(sp, 5, e)
        hist += np.bincount(arr["t"] // 3600, minlength=24)[:24]
        tot += len(arr)
    # expected share of hour h = integral of 1 + A cos(2 pi (t-39600)/86400) over the hour / 86400
    exp = np.array([3600 + A * 86400 / (2 * math.pi) * (math.sin(2 * math.pi * ((h + 1) * 3600 - 39600) / 86400)
                                                         - math.sin(2 * math.pi * (h * 3600 - 39600) / 86400)) for h in range(24)])
    exp = exp / 86400.0 * tot
    chi2 = float(((hist - exp) ** 2 / exp).sum())
    assert chi2 < 60.0, chi2                      # 23 dof: P(chi2 > 60) ~ 4e-5
    assert abs(tot - 120 * 1000) < 5 * math.sqrt(120 * 1000)
    assert hist[11] > 3.0 * hist[23]              # peak 11:00 vs trough 23:00 (ratio 4:1, PAPER.md:L286 peak hours)
    assert hist[5:17].sum() > hist[17:].sum() + hist[:5].sum()


def test_class_frequencies_and_slack_range():
    sp = _light_params(1000, 0.0, n_classes=4, weights=[4, 3, 2, 1])
    cls = []
    for e in range(40):
        r, arr = _arrivals(sp, 9, e)
        cls.append(arr["aux"].astype(np.int64))
        # due = t + floor(dur7 * slack / 1024), slack in [1536, 3072], dur7 in [1, 3]  ->  due - t in [1, 9]
        rel = arr["value"].astype(np.int64) - arr["t"].astype(np.int64)
        assert rel.min() >= 1 and rel.max() <= 9
    cls = np.concatenate(cls)
    freq = np.bincount(cls, minlength=4) / cls.size
    for f, w in zip(freq, [0.4, 0.3, 0.2, 0.1]):
        assert abs(f - w) < 4.5 * math.sqrt(w * (1 - w) / cls.size)


def test_slack_multiplier_uniform_between_1p5_and_3():
    # constant dur7 = 1000 s: rel = floor(1000 * slack / 1024) with slack uniform in [1536, 3072]
    sp = W.make_params([LINEAR], [W.dur_constant(1000)], [1], jobs_per_day=2000, amplitude=0.0, cap=1024, job_limit=0)
    rel = []
    for e in range(5):
        _, arr = _arrivals(sp, 2, e)
        rel.append(arr["value"].astype(np.int64) - arr["t"].astype(np.int64))
    rel = np.concatenate(rel)
    assert rel.min() >= 1500 and rel.max() <= 3000
    assert abs(rel.mean() - 2250.0) < 5 * (1500 / math.sqrt(12)) / math.sqrt(rel.size)
    assert rel.min() < 1530 and rel.max() > 2970


def test_episode_and_env_give_fresh_days_and_are_reproducible():
    sp = _light_params(300, 0.3)
    a = _arrivals(sp, 1, 0, 0)[0].totals["trace_hash"]
    assert a == _arrivals(sp, 1, 0, 0)[0].totals["trace_hash"]
    others = {int(_arrivals(sp, 1, 1, 0)[0].totals["trace_hash"]), int(_arrivals(sp, 1, 0, 1)[0].totals["trace_hash"]),
              int(_arrivals(sp, 2, 0, 0)[0].totals["trace_hash"]), int(_arrivals(sp, 1 << 32, 0, 0)[0].totals["trace_hash"])}
    assert int(a) not in others and len(others) == 4


def test_job_limit_reading_R6():
    sp = _light_params(300, 0.0, job_limit=50)
    r, arr = _arrivals(sp, 1, 0)
    assert len(arr) == 50 and int(r.totals["n_jobs"]) == 50


def test_md1_mean_wait_closed_form():
    """cfg 1 = single machine; one class, constant service D = 120 s, homogeneous Poisson
    lambda = 0.005/s (432/day), constant slack -> EDF == FCFS.  Pollaczek-Khinchine: W_q = rho D / (2 (1 - rho)) = 90 s."""
    D, lam = 120, 0.005
    sp = W.make_params([LINEAR], [W.dur_constant(D)], [1], jobs_per_day=lam * 86400, amplitude=0.0, slack=(2048, 2048),
                       cap=1024)
    waits, n = 0.0, 0
    n_env = 700                                   # ~300k jobs; sd of the mean wait estimate ~ 1 %
    for e in range(n_env):
        r = O.rollout(sp, 21, e, algo=0, cfg0=0, trace_cap=4000)
        tr = r.trace
        arr = {int(ev["job"]): int(ev["t"]) for ev in tr if ev["type"] == 1}
        assert int(r.totals["n_preempt"]) == 0    # FCFS: constant relative deadlines never reorder
        for ev in tr:
            if ev["type"] == 5:
                waits += int(ev["t"]) - arr[int(ev["job"])] - D
                n += 1
    mean_wait = waits / n
    # the day starts empty (transient) and integer ticks floor the arrival instant: allow 5 %
    assert abs(mean_wait - 90.0) < 4.5, mean_wait
