"""Seeded synthetic INPUT recipes for the batched MIG-day simulator (BASELINE.json configs C1..C5).

This module is the one thing the CPU oracle (``oracle/``) and the CUDA library
(``paper_2606_25082_b200/csrc``) have in common: it only *builds input arrays* (tables of
numbers handed identically to both sides).  It holds none of the method's arithmetic: no
Philox, no event loop, no scheduler, no power integration, no Q-network forward.  It imports
neither side.

Citations are PAPER.md line numbers (/root/reference/PAPER.md at authoring time) and
SURVEY.md section 8 rows.

* MIG configuration set: PAPER.md:L71-90 (Fig. 1), garbled rows 3/4 read as SURVEY 8(c.1).
* Job families linear / capped / sublinear: PAPER.md:L98-102, L222-224.
* Power: PAPER.md:L149-151 gives only a figure; BASELINE C1 gives "idle 30-60 W + dynamic
  proportional to slice^1.3" -> DESIGN.md reading #16.
* Arrivals: non-homogeneous Poisson process; peak hours 5:00-17:00 (L286);
  the sinusoid stands in for the paper's Fig. 5 (Alibaba-derived, not available).
"""
from __future__ import annotations

import dataclasses
import math
from statistics import NormalDist

import numpy as np

# --------------------------------------------------------------------------- constants
N_SLOTS = 7
SIZES = (1, 2, 3, 4, 7)           # slice sizes, index = "size index" used by every [..][5] table
SIZE_INDEX = {1: 0, 2: 1, 3: 2, 4: 3, 7: 4}
V7 = 840                           # work units per second on a 7g slice (divisible by 1..7)
STATE_DIM = 64
N_THR_BINS = 1440                  # one acceptance threshold per minute of the day

ALGO_EDF_FS, ALGO_EDF_SS, ALGO_LLF, ALGO_LALF, ALGO_EDF_SS_R = 0, 1, 2, 3, 4
ALGO_NAMES = ("EDF-FS", "EDF-SS", "LLF", "LALF", "EDF-SS-R")     # EDF-SS-R: restricted preemption
POLICY_STATIC, POLICY_TABLE, POLICY_DQN, POLICY_BINNED = 0, 1, 2, 3   # BINNED: table over the binned 2+2m state

# PAPER.md:L75-88 (Fig. 1): (size, start slot) per slice; config ids here are 0-based (paper id - 1).
FIG1_CONFIGS = (
    ((7, 0),),
    ((4, 0), (3, 4)),
    ((4, 0), (2, 4), (1, 6)),
    ((4, 0), (1, 4), (1, 5), (1, 6)),
    ((3, 0), (3, 4)),                                   # slot 3 is a hole
    ((2, 0), (2, 2), (3, 4)),
    ((2, 0), (1, 2), (1, 3), (3, 4)),
    ((1, 0), (1, 1), (1, 2), (1, 3), (3, 4)),
    ((2, 0), (2, 2), (2, 4), (1, 6)),
    ((2, 0), (2, 2), (1, 4), (1, 5), (1, 6)),
    ((2, 0), (1, 2), (1, 3), (1, 4), (1, 5), (1, 6)),
    ((1, 0), (1, 1), (1, 2), (1, 3), (1, 4), (1, 5), (1, 6)),
)


def size_at_slot_table(configs=FIG1_CONFIGS) -> np.ndarray:
    """[n_configs][7] u8: size of the slice STARTING at slot p, else 0."""
    out = np.zeros((len(configs), N_SLOTS), dtype=np.uint8)
    for c, row in enumerate(configs):
        for size, start in row:
            out[c, start] = size
    return out


# --------------------------------------------------------------------------- job families
def speed_linear() -> list[int]:
    """throughput proportional to slice size."""
    return [V7 * g // 7 for g in SIZES]


def speed_capped(k: int) -> list[int]:
    """linear up to a kg slice, flat after; 7g keeps the reference speed."""
    return [V7 * min(g, k) // k for g in SIZES]


def speed_sublinear(alpha: float) -> list[int]:
    """sublinear in slice size; BASELINE C1: exponent in U[0.5, 0.9]."""
    return [int(round(V7 * (g / 7.0) ** alpha)) for g in SIZES]


def dur_uniform(lo: float, hi: float) -> list[int]:
    """65-point quantile table of U[lo, hi] seconds on 7g."""
    return [max(1, int(round(lo + (hi - lo) * i / 64.0))) for i in range(65)]


def dur_constant(d: int) -> list[int]:
    return [int(d)] * 65


def dur_lognormal(median: float, sigma: float, clamp: int = 2_000_000) -> list[int]:
    """65-point quantile table of lognormal(ln median, sigma) (BASELINE C5 sigma=1.2)."""
    nd = NormalDist()
    q = []
    for i in range(65):
        z = nd.inv_cdf((i + 0.5) / 65.0)
        q.append(min(clamp, max(1, int(round(median * math.exp(sigma * z))))))
    return q


def table_mean(q: list[int]) -> float:
    """Mean of the piecewise-linear quantile table (for load targeting only)."""
    return float(np.mean([(q[i] + q[i + 1]) / 2.0 for i in range(64)]))


def class_cum_from_weights(w) -> np.ndarray:
    w = np.asarray(w, dtype=np.float64)
    c = np.cumsum(w) / np.sum(w)
    out = np.minimum(np.floor(c * 4294967296.0), 4294967295.0).astype(np.uint64)
    out[-1] = 0xFFFFFFFF
    return out.astype(np.uint32)


# --------------------------------------------------------------------------- power (reading #16)
def default_power():
    """p_idle[g] = 30000 + 5000(g-1) mW; p_busy[g] = p_idle[g] + round(15000 g^1.3) mW; curve = 0."""
    p_idle = [30000 + 5000 * (g - 1) for g in SIZES]
    p_busy = [pi + int(round(15000.0 * g ** 1.3)) for pi, g in zip(p_idle, SIZES)]
    return [0] * 8, p_idle, p_busy


# --------------------------------------------------------------------------- arrivals
def accept_thresholds(amplitude: float, peak_s: int = 39600) -> np.ndarray:
    """thr[b] = min(2^32-1, round(2^32 lambda(60b+30)/lambda_max)); lambda = 1 + A cos(2pi (t-peak)/86400).

    Peak 11:00, trough 23:00, positive half 5:00-17:00."""
    thr = np.empty(N_THR_BINS, dtype=np.uint32)
    for b in range(N_THR_BINS):
        t = 60 * b + 30
        lam = 1.0 + amplitude * math.cos(2.0 * math.pi * (t - peak_s) / 86400.0)
        v = int(round(4294967296.0 * lam / (1.0 + amplitude)))
        thr[b] = min(0xFFFFFFFF, max(0, v))
    return thr


def gap_scale_q16(jobs_per_day: float, amplitude: float) -> int:
    """C = round(2^16 ln2 / lambda_max), lambda_max = (1+A) N / 86400 per second."""
    lam_max = (1.0 + amplitude) * jobs_per_day / 86400.0
    return int(round(65536.0 * math.log(2.0) / lam_max))


# --------------------------------------------------------------------------- parameter bundle
@dataclasses.dataclass
class SimParams:
    speed: np.ndarray            # [n_classes][5] u32
    dur7_q: np.ndarray           # [n_classes][65] i32
    class_cum: np.ndarray        # [n_classes] u32
    slack_q10: np.ndarray        # [n_classes][2] u16
    size_at_slot: np.ndarray     # [n_configs][7] u8
    accept_thr: np.ndarray       # [1440] u32
    curve_mw: np.ndarray         # [8] i32
    p_idle_mw: np.ndarray        # [5] i32
    p_busy_mw: np.ndarray        # [5] i32
    gap_scale_q16: int
    day_s: int = 86400
    epoch_s: int = 3600
    n_epochs: int = 24
    t_limit_s: int = 2_592_000
    cap: int = 256
    job_limit: int = 0
    repart_downtime_s: int = 0
    repart_energy_mj: int = 0
    crit_laxity_s: int = 60
    crit_max: int = 3
    w_energy: float = 0.5
    w_tardy: float = 0.5
    env_offset: int = 0
    decide_on_events: int = 0    # TABLE / BINNED policy: also decide after every tick with an arrival or a completion
    # round-2 extensions (readings #29-#32); None / 0 = off
    speed_nomig: "np.ndarray | None" = None   # [n_classes] u32: work units / s on the whole GPU with MIG disabled (size code 8)
    p_idle_nomig_mw: int = 0
    p_busy_nomig_mw: int = 0
    repart_all_down: int = 0     # 1: a repartition takes the whole GPU down for repart_downtime_s
    gamma: float = 1.0           # discount of the return
    n_tbins: int = 0             # BINNED policy: time-of-day bins
    dbin_edges: "np.ndarray | None" = None    # [n_dbins - 1] i32 ascending edges of the deadline feature due - t (seconds)
    abin_edges: "np.ndarray | None" = None    # [n_abins - 1] i32 ascending edges of the mean remaining duration (seconds)
    util_hist: int = 0           # 1: keep the time spent per utilisation level (Fig. 6); CUDA side only (the oracle always does)

    @property
    def n_classes(self) -> int:
        return int(self.speed.shape[0])

    @property
    def n_configs(self) -> int:
        return int(self.size_at_slot.shape[0])

    @property
    def n_dbins(self) -> int:
        return 0 if self.dbin_edges is None else int(len(self.dbin_edges)) + 1

    @property
    def n_abins(self) -> int:
        return 0 if self.abin_edges is None else int(len(self.abin_edges)) + 1

    @property
    def binned_codes(self) -> int:
        """B = 1 + n_dbins * n_abins job codes per position (0 = no job); the BINNED table has n_configs * n_tbins * B^3 entries."""
        return 1 + self.n_dbins * self.n_abins

    def normalised(self) -> "SimParams":
        """Same values with the exact dtypes/contiguity both sides marshal from."""
        return dataclasses.replace(
            self,
            speed=np.ascontiguousarray(self.speed, dtype=np.uint32),
            dur7_q=np.ascontiguousarray(self.dur7_q, dtype=np.int32),
            class_cum=np.ascontiguousarray(self.class_cum, dtype=np.uint32),
            slack_q10=np.ascontiguousarray(self.slack_q10, dtype=np.uint16),
            size_at_slot=np.ascontiguousarray(self.size_at_slot, dtype=np.uint8),
            accept_thr=np.ascontiguousarray(self.accept_thr, dtype=np.uint32),
            curve_mw=np.ascontiguousarray(self.curve_mw, dtype=np.int32),
            p_idle_mw=np.ascontiguousarray(self.p_idle_mw, dtype=np.int32),
            p_busy_mw=np.ascontiguousarray(self.p_busy_mw, dtype=np.int32),
            speed_nomig=None if self.speed_nomig is None else np.ascontiguousarray(self.speed_nomig, dtype=np.uint32),
            dbin_edges=None if self.dbin_edges is None else np.ascontiguousarray(self.dbin_edges, dtype=np.int32),
            abin_edges=None if self.abin_edges is None else np.ascontiguousarray(self.abin_edges, dtype=np.int32),
        )


def make_params(speeds, durs, weights, *, jobs_per_day, amplitude, slack=(1536, 3072),
                configs=FIG1_CONFIGS, **kw) -> SimParams:
    curve, p_idle, p_busy = default_power()
    n = len(speeds)
    return SimParams(
        speed=np.array(speeds, dtype=np.uint32).reshape(n, 5),
        dur7_q=np.array(durs, dtype=np.int32).reshape(n, 65),
        class_cum=class_cum_from_weights(weights),
        slack_q10=np.array([slack] * n, dtype=np.uint16),
        size_at_slot=size_at_slot_table(configs),
        accept_thr=accept_thresholds(amplitude),
        curve_mw=np.array(curve, dtype=np.int32),
        p_idle_mw=np.array(p_idle, dtype=np.int32),
        p_busy_mw=np.array(p_busy, dtype=np.int32),
        gap_scale_q16=gap_scale_q16(jobs_per_day, amplitude),
        **kw,
    ).normalised()


@dataclasses.dataclass
class QNetWeights:
    """MLP 64-256-256-n_actions, fp32, W stored [in][out] row-major."""
    W1: np.ndarray
    b1: np.ndarray
    W2: np.ndarray
    b2: np.ndarray
    W3: np.ndarray
    b3: np.ndarray

    @property
    def n_actions(self) -> int:
        return int(self.W3.shape[1])


def make_qnet(seed: int, n_actions: int = 12, hidden: int = 256) -> QNetWeights:
    """Seed-initialised weights U(-1/sqrt(fan_in), +1/sqrt(fan_in)); no trained weights exist."""
    rng = np.random.default_rng(seed)

    def layer(fi, fo):
        b = 1.0 / math.sqrt(fi)
        return (rng.uniform(-b, b, size=(fi, fo)).astype(np.float32),
                rng.uniform(-b, b, size=(fo,)).astype(np.float32))

    W1, b1 = layer(STATE_DIM, hidden)
    W2, b2 = layer(hidden, hidden)
    W3, b3 = layer(hidden, n_actions)
    return QNetWeights(W1, b1, W2, b2, W3, b3)


@dataclasses.dataclass
class Workload:
    name: str
    params: SimParams
    n_envs: int
    seed: int
    algo: np.ndarray             # [n_envs] u8
    cfg0: np.ndarray             # [n_envs] u8
    policy: int
    table: np.ndarray | None = None      # [n_envs][n_epochs][4] u8
    qnet: QNetWeights | None = None
    epsilon: float = 0.0
    mean_jobs_per_day: float = 0.0


# --------------------------------------------------------------------------- the five BASELINE configs
_FAMILIES8 = (
    ("linear", speed_linear()),
    ("sub0.5", speed_sublinear(0.5)),
    ("sub0.6", speed_sublinear(0.6)),
    ("sub0.75", speed_sublinear(0.75)),
    ("sub0.9", speed_sublinear(0.9)),
    ("cap2", speed_capped(2)),
    ("cap3", speed_capped(3)),
    ("cap4", speed_capped(4)),
)


def config_c1(n_envs: int = 1) -> Workload:
    """BASELINE C1: 1 env, static {3g,2g,1g,1g} (Fig. 1 config 7), 3 sublinear classes with constant
    dur7 in U[60,3600] and exponent in U[0.5,0.9], homogeneous Poisson 200/day, seed 0."""
    rng = np.random.default_rng(1000)
    alphas = rng.uniform(0.5, 0.9, size=3)
    durs = rng.integers(60, 3601, size=3)
    p = make_params([speed_sublinear(float(a)) for a in alphas], [dur_constant(int(d)) for d in durs],
                    [1, 1, 1], jobs_per_day=200, amplitude=0.0, cap=256)
    return Workload("C1", p, n_envs, 0, np.full(n_envs, ALGO_EDF_SS, np.uint8), np.full(n_envs, 6, np.uint8),
                    POLICY_STATIC, mean_jobs_per_day=200)


def config_c2(n_envs: int = 1024) -> Workload:
    """BASELINE C2: diurnal 4:1 (A=0.6), 2000 jobs/day, 8 classes (paper's families), each of the 4
    algorithms x each of the 12 Fig. 1 partitions held static, preemption on, w=0.5."""
    p = make_params([s for _, s in _FAMILIES8], [dur_uniform(2, 37)] * 8, [1] * 8,
                    jobs_per_day=2000, amplitude=0.6, cap=256)
    e = np.arange(n_envs)
    return Workload("C2", p, n_envs, 1, (e % 4).astype(np.uint8), ((e // 4) % 12).astype(np.uint8),
                    POLICY_STATIC, mean_jobs_per_day=2000)


def _classes12():
    fams = (speed_linear(), speed_sublinear(0.5), speed_sublinear(0.7), speed_sublinear(0.9),
            speed_capped(2), speed_capped(4))
    speeds, durs, w = [], [], []
    for f in fams:                      # short "inference-like" 80 %, long "training-like" 20 %
        speeds.append(f); durs.append(dur_uniform(2, 20)); w.append(0.8)
        speeds.append(f); durs.append(dur_uniform(30, 150)); w.append(0.2)
    return speeds, durs, w


def _twice_daily_table(n_envs: int, n_cfg: int, rng) -> tuple[np.ndarray, np.ndarray]:
    a = rng.integers(0, n_cfg, size=n_envs)
    b = (a + 1 + rng.integers(0, n_cfg - 1, size=n_envs)) % n_cfg       # uniform among the rest
    table = np.empty((n_envs, 24, 4), dtype=np.uint8)
    for h in range(24):
        table[:, h, :] = np.where((h >= 8) & (h < 20), b, a)[:, None]
    return table, a.astype(np.uint8)


def config_c3(n_envs: int = 4096) -> Workload:
    """BASELINE C3: twice-daily repartitioning (08:00/20:00) between two seeded-random valid partitions,
    60 s downtime of affected slices + fixed energy, queue cap 256, 12 classes."""
    speeds, durs, w = _classes12()
    p = make_params(speeds, durs, w, jobs_per_day=2000, amplitude=0.6, cap=256,
                    repart_downtime_s=60, repart_energy_mj=6_000_000)
    table, cfg0 = _twice_daily_table(n_envs, 12, np.random.default_rng(1002))
    return Workload("C3", p, n_envs, 2, np.full(n_envs, ALGO_EDF_SS, np.uint8), cfg0, POLICY_TABLE,
                    table=table, mean_jobs_per_day=2000)


def config_c4(n_envs: int = 8192) -> Workload:
    """BASELINE C4: DQN-driven repartitioning at 24 hourly epochs, MLP 64-256-256-12, eps=0.1;
    repartition penalty = the paper's 4 s."""
    speeds, durs, w = _classes12()
    p = make_params(speeds, durs, w, jobs_per_day=2000, amplitude=0.6, cap=256,
                    repart_downtime_s=4, repart_energy_mj=0)
    cfg0 = (np.arange(n_envs) % 12).astype(np.uint8)
    return Workload("C4", p, n_envs, 3, np.full(n_envs, ALGO_EDF_SS, np.uint8), cfg0, POLICY_DQN,
                    qnet=make_qnet(1003, 12), epsilon=0.1, mean_jobs_per_day=2000)


def _c5_table(n_envs: int) -> np.ndarray:
    """Fixed tabulated policy [24][4] (bucket by jobs in system): nights cfg 2, days alternate cfg 3 / cfg 6,
    heavy backlog (bucket 3) -> cfg 1 by day, cfg 2 by night; empty system keeps cfg 2 (paper ids)."""
    t = np.empty((24, 4), dtype=np.uint8)
    for h in range(24):
        day = 5 <= h < 17                                   # PAPER.md:L286 peak hours
        base = (2 if h % 2 == 0 else 5) if day else 1       # 0-based ids of cfg 3 / cfg 6 / cfg 2
        t[h] = (1, base, base, 0 if day else 1)
    return np.broadcast_to(t, (n_envs, 24, 4)).copy()


def config_c5(n_envs: int = 65536) -> Workload:
    """BASELINE C5: heavy load 8000 jobs/day, peak/trough 6:1 (A=5/7), 16 classes with lognormal(sigma=1.2)
    runtimes, queue cap 1024, preemption + hourly repartitioning from a fixed tabulated policy."""
    speeds, durs, w = [], [], []
    med = 1.75                                             # chosen so that rho_7 = N E[dur7] / 86400 ~ 0.75
    for _, f in _FAMILIES8:
        speeds.append(f); durs.append(dur_lognormal(med, 1.2)); w.append(0.8)
        speeds.append(f); durs.append(dur_lognormal(8 * med, 1.2)); w.append(0.2)
    p = make_params(speeds, durs, w, jobs_per_day=8000, amplitude=5.0 / 7.0, cap=1024,
                    repart_downtime_s=60, repart_energy_mj=6_000_000)
    return Workload("C5", p, n_envs, 4, np.full(n_envs, ALGO_EDF_SS, np.uint8), np.full(n_envs, 1, np.uint8),
                    POLICY_TABLE, table=_c5_table(n_envs), mean_jobs_per_day=8000)


# --------------------------------------------------------------------------- the paper's benchmark policies and sweeps
# (SURVEY 8(f) #4).  Input recipes only: tables, no arithmetic of the method.
NOMIG_CONFIG = ((8, 0),)             # size code 8 = the whole GPU with MIG disabled (reading #29)
PAPER_STATIC_CFG, PAPER_DAY_CFG, PAPER_NIGHT_CFG = 2, 5, 1     # 0-based ids of the paper's configurations 3, 6 and 2 (L230)


def speed_nomig_of(speeds) -> np.ndarray:
    """Speed on the MIG-disabled GPU per class: "6% performance improvement for linear jobs ... compared to a 7g.40gb slice"
    (PAPER.md:L230): round(1.06 v_7g) for the linear family, v_7g for every other (the paper names linear jobs only)."""
    lin = speed_linear()
    return np.array([int(round(1.06 * s[4])) if list(s) == lin else int(s[4]) for s in speeds], dtype=np.uint32)


def benchmark_params(jobs_per_day=2000.0, amplitude=0.6, inference_frac=0.8, **kw) -> SimParams:
    """The C3/C4 class mix (6 elasticity families x short "inference-like" / long "training-like")
    with the 12 configurations of Fig. 1 plus the MIG-disabled GPU as a 13th (id 12), the paper's 4 s repartition
    penalty for the whole GPU (L214), the discount of its reward model and the utilisation levels of Fig. 6."""
    fams = (speed_linear(), speed_sublinear(0.5), speed_sublinear(0.7), speed_sublinear(0.9), speed_capped(2), speed_capped(4))
    speeds, durs, w = [], [], []
    for f in fams:
        speeds.append(f); durs.append(dur_uniform(2, 20)); w.append(inference_frac)
        speeds.append(f); durs.append(dur_uniform(30, 150)); w.append(1.0 - inference_frac)
    args = dict(cap=256, repart_downtime_s=4, repart_energy_mj=0)
    args.update(kw)
    p = make_params(speeds, durs, w, jobs_per_day=jobs_per_day, amplitude=amplitude, configs=FIG1_CONFIGS + (NOMIG_CONFIG,), **args)
    curve, p_idle, p_busy = default_power()
    return dataclasses.replace(p, speed_nomig=speed_nomig_of(speeds), p_idle_nomig_mw=p_idle[4], p_busy_nomig_mw=p_busy[4],
                               repart_all_down=1, gamma=0.99, util_hist=1)


def day_night_table(n_envs: int) -> np.ndarray:
    """"Configuration 6 for day-time, defined as 5:00-17:00, and Configuration 2 for night-time"."""
    t = np.empty((24, 4), dtype=np.uint8)
    for h in range(24):
        t[h] = PAPER_DAY_CFG if 5 <= h < 17 else PAPER_NIGHT_CFG
    return np.broadcast_to(t, (n_envs, 24, 4)).copy()


def config_benchmark(kind: str, n_envs: int = 1024, algo: int = ALGO_EDF_SS_R, **kw) -> Workload:
    """The paper's three benchmark policies (L230) on one parameter set: "nomig" (full GPU, MIG disabled), "static"
    (configuration 3), "daynight" (configuration 6 from 5:00 to 17:00, configuration 2 otherwise).  The dynamic policy is
    C4 (DQN) / the BINNED policy.  algo defaults to EDF-SS with restricted preemption, which the paper's repartitioning
    experiments run on (L198-204)."""
    p = benchmark_params(**kw)
    a = np.full(n_envs, algo, np.uint8)
    if kind == "nomig":
        return Workload("nomig", p, n_envs, 11, a, np.full(n_envs, 12, np.uint8), POLICY_STATIC, mean_jobs_per_day=2000)
    if kind == "static":
        return Workload("static", p, n_envs, 11, a, np.full(n_envs, PAPER_STATIC_CFG, np.uint8), POLICY_STATIC, mean_jobs_per_day=2000)
    if kind == "daynight":
        return Workload("daynight", p, n_envs, 11, a, np.full(n_envs, PAPER_NIGHT_CFG, np.uint8), POLICY_TABLE,
                        table=day_night_table(n_envs), mean_jobs_per_day=2000)
    raise ValueError(kind)


# The sweeps of Figs. 7-10 are parameter files: the arrival rates 0.1 / 0.5 / 0.75 of L240 relative to the default 0.5,
# the 20 % / 80 % inference split of L242.
SWEEP_RATE_SCALE = {"0.1": 0.2, "0.5": 1.0, "0.75": 1.5}
SWEEP_INFERENCE = {"20": 0.2, "80": 0.8}


def binned_defaults(p: SimParams) -> SimParams:
    """Bin edges of the BINNED policy's state (PAPER.md:L210 gives none; reading #31): 24 hourly time bins,
    deadline bins overdue | within 10 min | later, average-duration bins < 30 s | < 300 s | longer."""
    return dataclasses.replace(p, n_tbins=24, dbin_edges=np.array([0, 600], dtype=np.int32), abin_edges=np.array([30, 300], dtype=np.int32))


CONFIGS = {"C1": config_c1, "C2": config_c2, "C3": config_c3, "C4": config_c4, "C5": config_c5}


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Env-range partition for data-parallel sharding: rank r gets [lo, hi)."""
    lo = (n_total * rank) // world
    hi = (n_total * (rank + 1)) // world
    return lo, hi


def reduce_over_ranks(seconds: float, units: int, device="cpu") -> tuple[float, int]:
    """Whole-job timing of a data-parallel run: the slowest rank's time and the units of all ranks.  Works
    on any initialised torch.distributed backend (NCCL with a CUDA device, gloo on CPU); a no-op without one."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(seconds), int(units)
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    n = torch.tensor([units], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), int(n.item())
