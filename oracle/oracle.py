"""ctypes front end of the CPU oracle (oracle/mig_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package's binding; inputs come as plain numpy arrays / the SimParams dataclass
from ``paper_2606_25082_b200.workloads`` (input recipes only).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

STATE_DIM = 64

EVENT_DTYPE = np.dtype([("t", "<i4"), ("type", "u1"), ("slot", "u1"), ("aux", "<u2"), ("job", "<u4"), ("value", "<i4")])
REC_DTYPE = np.dtype([
    ("energy_mj", "<i8"), ("tardiness_s", "<i8"), ("trace_hash", "<u8"), ("busy_unit_s", "<i4"), ("t_end", "<i4"),
    ("n_events", "<u4"), ("n_arrived", "<u2"), ("n_completed", "<u2"), ("n_dropped", "<u2"), ("n_tardy", "<u2"),
    ("n_preempt", "<u2"), ("n_start", "<u2"), ("n_crit", "<u2"), ("n_sys_end", "<u2"), ("cfg", "u1"),
    ("repartitioned", "u1"), ("status", "u1"), ("n_running_end", "u1"), ("n_sys_max", "<u4"), ("pad_", "<u4")])
TOTALS_DTYPE = np.dtype([
    ("energy_mj", "<i8"), ("tardiness_s", "<i8"), ("trace_hash", "<u8"), ("busy_unit_s", "<i8"), ("n_jobs", "<u4"),
    ("n_completed", "<u4"), ("n_dropped", "<u4"), ("n_tardy", "<u4"), ("n_preempt", "<u4"), ("n_start", "<u4"),
    ("n_crit", "<u4"), ("n_events", "<u4"), ("n_repart", "<u4"), ("n_sys_max", "<u4"), ("t_end", "<i4"),
    ("status", "<u4")])
JOB_IN_DTYPE = np.dtype([("arr", "<i4"), ("cls", "<u4"), ("dur7", "<i4"), ("due", "<i4")])
assert EVENT_DTYPE.itemsize == 16 and REC_DTYPE.itemsize == 64 and TOTALS_DTYPE.itemsize == 80

EV_ARRIVE, EV_DROP, EV_START, EV_PREEMPT, EV_COMPLETE, EV_CRIT, EV_SLICE_UP, EV_REPART = range(1, 9)
ST_TRUNCATED, ST_BAD_ACTION, ST_BAD_ALGO = 1, 2, 4


class _Params(C.Structure):
    _fields_ = [
        ("n_classes", C.c_uint32), ("n_configs", C.c_uint32),
        ("speed", C.c_void_p), ("dur7_q", C.c_void_p), ("class_cum", C.c_void_p), ("slack_q10", C.c_void_p),
        ("size_at_slot", C.c_void_p), ("accept_thr", C.c_void_p),
        ("curve_mw", C.c_int32 * 8), ("p_idle_mw", C.c_int32 * 5), ("p_busy_mw", C.c_int32 * 5),
        ("gap_scale_q16", C.c_uint64),
        ("day_s", C.c_int32), ("epoch_s", C.c_int32), ("n_epochs", C.c_int32), ("t_limit_s", C.c_int32),
        ("cap", C.c_uint32), ("job_limit", C.c_uint32),
        ("repart_downtime_s", C.c_int32), ("repart_energy_mj", C.c_int64),
        ("crit_laxity_s", C.c_int32), ("crit_max", C.c_uint32),
        ("w_energy", C.c_float), ("w_tardy", C.c_float),
        ("decide_on_events", C.c_uint32),
        ("speed_nomig", C.c_void_p), ("p_idle_nomig_mw", C.c_int32), ("p_busy_nomig_mw", C.c_int32),
        ("repart_all_down", C.c_uint32), ("gamma", C.c_float),
        ("n_tbins", C.c_uint32), ("n_dbins", C.c_uint32), ("n_abins", C.c_uint32),
        ("dbin_edges", C.c_void_p), ("abin_edges", C.c_void_p),
    ]


class _QNet(C.Structure):
    _fields_ = [("n_actions", C.c_uint32), ("hidden", C.c_uint32),
                ("W1", C.c_void_p), ("b1", C.c_void_p), ("W2", C.c_void_p), ("b2", C.c_void_p),
                ("W3", C.c_void_p), ("b3", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        # MIG_ORACLE_LIB: an alternative build of the same source (tests/test_oracle_sanitizers.py: ASan + UBSan)
        _lib = C.CDLL(os.environ.get("MIG_ORACLE_LIB") or _build.build())
        _lib.orc_neglog2_q24.restype = C.c_uint32
        _lib.orc_neglog2_q24.argtypes = [C.c_uint32]
        _lib.orc_fnv1a_words.restype = C.c_uint64
        _lib.orc_fnv1a_words.argtypes = [C.c_uint64, C.c_void_p]
        _lib.orc_env_create.restype = C.c_void_p
        _lib.orc_env_create.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32]
        _lib.orc_env_destroy.argtypes = [C.c_void_p]
        _lib.orc_env_set_jobs.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32]
        _lib.orc_env_set_trace.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32]
        _lib.orc_env_reset.argtypes = [C.c_void_p, C.c_uint32, C.c_uint8, C.c_uint8]
        _lib.orc_env_step.restype = C.c_int
        _lib.orc_env_step.argtypes = [C.c_void_p, C.c_uint8, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.orc_env_observe.argtypes = [C.c_void_p, C.c_void_p]
        _lib.orc_env_totals.argtypes = [C.c_void_p, C.c_void_p]
        _lib.orc_env_n_sys.restype = C.c_uint32
        _lib.orc_env_n_sys.argtypes = [C.c_void_p]
        _lib.orc_rollout.restype = C.c_int
        _lib.orc_rollout.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint8, C.c_uint8, C.c_int,
                                     C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.orc_rollout_ex.restype = C.c_int
        _lib.orc_rollout_ex.argtypes = _lib.orc_rollout.argtypes + [C.c_void_p, C.c_void_p]
        _lib.orc_env_binned_index.restype = C.c_uint32
        _lib.orc_env_binned_index.argtypes = [C.c_void_p]
        _lib.orc_env_util_hist.argtypes = [C.c_void_p, C.c_void_p]
        _lib.orc_et_reduce.restype = C.c_double
        _lib.orc_et_reduce.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]
        _lib.orc_dqn_n_params.restype = C.c_size_t
        _lib.orc_dqn_n_params.argtypes = [C.c_uint32, C.c_uint32]
        _lib.orc_dqn_create.restype = C.c_void_p
        _lib.orc_dqn_create.argtypes = [C.c_void_p, C.c_double, C.c_double]
        _lib.orc_dqn_destroy.argtypes = [C.c_void_p]
        _lib.orc_dqn_sync_target.argtypes = [C.c_void_p]
        _lib.orc_dqn_get.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        _lib.orc_dqn_set.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        _lib.orc_dqn_q.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_uint32, C.c_void_p]
        _lib.orc_dqn_loss_grad.restype = C.c_double
        _lib.orc_dqn_loss_grad.argtypes = [C.c_void_p] * 6 + [C.c_uint32, C.c_void_p]
        _lib.orc_dqn_train_step.restype = C.c_double
        _lib.orc_dqn_train_step.argtypes = [C.c_void_p] * 6 + [C.c_uint32]
        _lib.orc_replay_sample.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p]
        _lib.orc_q_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p]
        _lib.orc_q_eval_f64.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
        _lib.orc_philox4x32_10.argtypes = [C.c_uint32] * 6 + [C.c_void_p]
        _lib.orc_log_table.argtypes = [C.c_void_p]
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class ParamsHolder:
    """Marshals a workloads.SimParams into the oracle's C struct, keeping the arrays alive."""

    def __init__(self, sp):
        sp = sp.normalised()
        self.sp = sp
        s = _Params()
        s.n_classes, s.n_configs = sp.n_classes, sp.n_configs
        self._keep = (sp.speed, sp.dur7_q, sp.class_cum, sp.slack_q10, sp.size_at_slot, sp.accept_thr)
        s.speed, s.dur7_q, s.class_cum = _ptr(sp.speed), _ptr(sp.dur7_q), _ptr(sp.class_cum)
        s.slack_q10, s.size_at_slot, s.accept_thr = _ptr(sp.slack_q10), _ptr(sp.size_at_slot), _ptr(sp.accept_thr)
        for i in range(8):
            s.curve_mw[i] = int(sp.curve_mw[i])
        for i in range(5):
            s.p_idle_mw[i] = int(sp.p_idle_mw[i])
            s.p_busy_mw[i] = int(sp.p_busy_mw[i])
        s.gap_scale_q16 = int(sp.gap_scale_q16)
        s.day_s, s.epoch_s, s.n_epochs, s.t_limit_s = sp.day_s, sp.epoch_s, sp.n_epochs, sp.t_limit_s
        s.cap, s.job_limit = sp.cap, sp.job_limit
        s.repart_downtime_s, s.repart_energy_mj = sp.repart_downtime_s, sp.repart_energy_mj
        s.crit_laxity_s, s.crit_max = sp.crit_laxity_s, sp.crit_max
        s.w_energy, s.w_tardy = sp.w_energy, sp.w_tardy
        s.decide_on_events = int(getattr(sp, "decide_on_events", 0))
        self._keep2 = (sp.speed_nomig, sp.dbin_edges, sp.abin_edges)
        s.speed_nomig = _ptr(sp.speed_nomig)
        s.p_idle_nomig_mw, s.p_busy_nomig_mw = int(sp.p_idle_nomig_mw), int(sp.p_busy_nomig_mw)
        s.repart_all_down, s.gamma = int(sp.repart_all_down), float(sp.gamma)
        s.n_tbins, s.n_dbins, s.n_abins = int(sp.n_tbins), int(sp.n_dbins), int(sp.n_abins)
        s.dbin_edges, s.abin_edges = _ptr(sp.dbin_edges), _ptr(sp.abin_edges)
        self.c = s

    @property
    def ref(self):
        return C.byref(self.c)


class QNetHolder:
    def __init__(self, qw):
        self.arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (qw.W1, qw.b1, qw.W2, qw.b2, qw.W3, qw.b3)]
        q = _QNet()
        q.n_actions, q.hidden = int(self.arrs[4].shape[1]), int(self.arrs[0].shape[1])
        q.W1, q.b1, q.W2, q.b2, q.W3, q.b3 = (_ptr(a) for a in self.arrs)
        self.c = q
        self.n_actions = q.n_actions

    @property
    def ref(self):
        return C.byref(self.c)


def philox(c0, c1, c2, c3, k0, k1) -> np.ndarray:
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c0, c1, c2, c3, k0, k1, _ptr(out))
    return out


def neglog2_q24(w: int) -> int:
    return int(lib().orc_neglog2_q24(w))


def log_table() -> np.ndarray:
    out = np.zeros(257, dtype=np.uint32)
    lib().orc_log_table(_ptr(out))
    return out


def fnv1a_words(h: int, words) -> int:
    w = np.asarray(words, dtype=np.uint32)
    return int(lib().orc_fnv1a_words(h, _ptr(w)))


def make_jobs(rows) -> np.ndarray:
    """rows: iterable of (arr, cls, dur7, due)."""
    a = np.zeros(len(rows), dtype=JOB_IN_DTYPE)
    for i, r in enumerate(rows):
        a[i] = tuple(r)
    return a


class RolloutResult:
    __slots__ = ("recs", "totals", "trace", "states", "actions", "rewards", "ret", "util")


def rollout(sp, seed, env_id, *, episode=0, algo=1, cfg0=0, policy=0, table=None, qnet=None, epsilon=0.0,
            jobs=None, trace_cap=0, want_states=False) -> RolloutResult:
    """One env-day on the oracle.  ``table``: [n_epochs][4] u8 for THIS env; ``qnet``: workloads.QNetWeights."""
    ph = sp if isinstance(sp, ParamsHolder) else ParamsHolder(sp)
    ne = ph.sp.n_epochs
    recs = np.zeros(ne + 1, dtype=REC_DTYPE)
    totals = np.zeros(1, dtype=TOTALS_DTYPE)
    trace = np.zeros(trace_cap, dtype=EVENT_DTYPE) if trace_cap else None
    ntr = np.zeros(1, dtype=np.uint32)
    states = np.zeros((ne + 1, STATE_DIM), dtype=np.float32) if want_states else None
    actions = np.zeros(ne, dtype=np.uint8)
    rewards = np.zeros(ne, dtype=np.float32)
    tb = None if table is None else np.ascontiguousarray(table, dtype=np.uint8)
    qh = None if qnet is None else (qnet if isinstance(qnet, QNetHolder) else QNetHolder(qnet))
    jb = None if jobs is None else np.ascontiguousarray(jobs, dtype=JOB_IN_DTYPE)
    ret = np.zeros(1, dtype=np.float32)
    util = np.zeros(8, dtype=np.int32)
    rc = lib().orc_rollout_ex(ph.ref, seed, env_id, episode, algo, cfg0, policy, _ptr(tb), qh.ref if qh else None,
                              epsilon, _ptr(jb), 0 if jb is None else len(jb), _ptr(recs), _ptr(totals), _ptr(trace),
                              trace_cap, _ptr(ntr), _ptr(states), _ptr(actions), _ptr(rewards), _ptr(ret), _ptr(util))
    assert rc == 0
    r = RolloutResult()
    r.ret, r.util = float(ret[0]), util
    r.recs, r.totals = recs, totals[0]
    if trace is not None:
        assert ntr[0] <= trace_cap, "trace buffer too small: %d events" % ntr[0]
        r.trace = trace[: ntr[0]]
    else:
        r.trace = None
    r.states, r.actions, r.rewards = states, actions, rewards
    return r


class Env:
    """Step-wise access to one oracle environment."""

    def __init__(self, sp, seed, env_id, jobs=None, trace_cap=0):
        self.ph = sp if isinstance(sp, ParamsHolder) else ParamsHolder(sp)
        self.h = lib().orc_env_create(self.ph.ref, seed, env_id)
        self._jobs = None
        if jobs is not None:
            self._jobs = np.ascontiguousarray(jobs, dtype=JOB_IN_DTYPE)
            lib().orc_env_set_jobs(self.h, _ptr(self._jobs), len(self._jobs))
        self.trace_buf = np.zeros(trace_cap, dtype=EVENT_DTYPE) if trace_cap else None
        if trace_cap:
            lib().orc_env_set_trace(self.h, _ptr(self.trace_buf), trace_cap)

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_env_destroy(self.h)
            self.h = None

    def reset(self, episode=0, algo=1, cfg0=0):
        lib().orc_env_reset(self.h, episode, algo, cfg0)
        return self.observe()

    def observe(self):
        x = np.zeros(STATE_DIM, dtype=np.float32)
        lib().orc_env_observe(self.h, _ptr(x))
        return x

    def step(self, action):
        x = np.zeros(STATE_DIM, dtype=np.float32)
        r = np.zeros(1, dtype=np.float32)
        dE = np.zeros(1, dtype=np.int64)
        dT = np.zeros(1, dtype=np.int64)
        rec = np.zeros(2, dtype=REC_DTYPE)
        rc = lib().orc_env_step(self.h, action, _ptr(x), _ptr(r), _ptr(dE), _ptr(dT), _ptr(rec))
        if rc != 0:
            raise RuntimeError("day is over")
        return x, float(r[0]), int(dE[0]), int(dT[0]), rec

    def totals(self):
        t = np.zeros(1, dtype=TOTALS_DTYPE)
        lib().orc_env_totals(self.h, _ptr(t))
        return t[0]

    def n_sys(self):
        return int(lib().orc_env_n_sys(self.h))

    def binned_index(self):
        return int(lib().orc_env_binned_index(self.h))

    def util_hist(self):
        u = np.zeros(8, dtype=np.int32)
        lib().orc_env_util_hist(self.h, _ptr(u))
        return u

    def trace(self):
        n = int(self.totals()["n_events"])
        assert n <= len(self.trace_buf)
        return self.trace_buf[:n]


def q_eval(qnet, states):
    qh = qnet if isinstance(qnet, QNetHolder) else QNetHolder(qnet)
    x = np.ascontiguousarray(states, dtype=np.float32).reshape(-1, STATE_DIM)
    q = np.zeros((x.shape[0], qh.n_actions), dtype=np.float32)
    am = np.zeros(x.shape[0], dtype=np.uint8)
    lib().orc_q_eval(qh.ref, _ptr(x), x.shape[0], _ptr(q), _ptr(am))
    return q, am


def q_eval_f64(qnet, states):
    qh = qnet if isinstance(qnet, QNetHolder) else QNetHolder(qnet)
    x = np.ascontiguousarray(states, dtype=np.float32).reshape(-1, STATE_DIM)
    q = np.zeros((x.shape[0], qh.n_actions), dtype=np.float64)
    lib().orc_q_eval_f64(qh.ref, _ptr(x), x.shape[0], _ptr(q))
    return q


def et_reduce(x, y, group, n_groups):
    """ET per group and the global scaling factor a."""
    x = np.ascontiguousarray(x, dtype=np.float64); y = np.ascontiguousarray(y, dtype=np.float64)
    g = np.ascontiguousarray(group, dtype=np.uint32)
    et = np.zeros(n_groups, dtype=np.float64)
    a = lib().orc_et_reduce(_ptr(x), _ptr(y), _ptr(g), len(x), n_groups, _ptr(et))
    return et, float(a)


class Dqn:
    """The DQN training oracle (dqn_oracle.c): online + frozen target network in double precision, squared TD error, SGD."""

    def __init__(self, qnet, gamma: float, lr: float):
        qh = qnet if isinstance(qnet, QNetHolder) else QNetHolder(qnet)
        self.H, self.A = int(qh.c.hidden), int(qh.c.n_actions)
        self.n = int(lib().orc_dqn_n_params(self.H, self.A))
        self.h = lib().orc_dqn_create(qh.ref, float(gamma), float(lr))

    def __del__(self):
        if getattr(self, "h", None):
            lib().orc_dqn_destroy(self.h)
            self.h = None

    @staticmethod
    def _batch(s, a, r, s2, done):
        s = np.ascontiguousarray(s, dtype=np.float32).reshape(-1, STATE_DIM)
        s2 = np.ascontiguousarray(s2, dtype=np.float32).reshape(-1, STATE_DIM)
        a = np.ascontiguousarray(a, dtype=np.uint8); r = np.ascontiguousarray(r, dtype=np.float32)
        done = np.zeros(len(a), np.uint8) if done is None else np.ascontiguousarray(done, dtype=np.uint8)
        assert len(s) == len(s2) == len(a) == len(r) == len(done)
        return s, a, r, s2, done

    def params(self, which=0) -> np.ndarray:
        out = np.zeros(self.n, dtype=np.float64)
        lib().orc_dqn_get(self.h, which, _ptr(out))
        return out

    def set_params(self, flat, which=0):
        f = np.ascontiguousarray(flat, dtype=np.float64)
        assert f.size == self.n
        lib().orc_dqn_set(self.h, which, _ptr(f))

    def split(self, flat):
        """flat -> (W1 [64][H], b1, W2 [H][H], b2, W3 [H][A], b3)"""
        H, A = self.H, self.A
        sz = [STATE_DIM * H, H, H * H, H, H * A, A]
        sh = [(STATE_DIM, H), (H,), (H, H), (H,), (H, A), (A,)]
        out, o = [], 0
        for n, shp in zip(sz, sh):
            out.append(np.asarray(flat[o:o + n]).reshape(shp)); o += n
        return out

    def q(self, s, which=0) -> np.ndarray:
        s = np.ascontiguousarray(s, dtype=np.float32).reshape(-1, STATE_DIM)
        out = np.zeros((len(s), self.A), dtype=np.float64)
        lib().orc_dqn_q(self.h, which, _ptr(s), len(s), _ptr(out))
        return out

    def loss_grad(self, s, a, r, s2, done=None, want_grad=True):
        s, a, r, s2, done = self._batch(s, a, r, s2, done)
        g = np.zeros(self.n, dtype=np.float64) if want_grad else None
        loss = lib().orc_dqn_loss_grad(self.h, _ptr(s), _ptr(a), _ptr(r), _ptr(s2), _ptr(done), len(a), _ptr(g))
        return float(loss), g

    def train_step(self, s, a, r, s2, done=None) -> float:
        s, a, r, s2, done = self._batch(s, a, r, s2, done)
        return float(lib().orc_dqn_train_step(self.h, _ptr(s), _ptr(a), _ptr(r), _ptr(s2), _ptr(done), len(a)))

    def sync_target(self):
        lib().orc_dqn_sync_target(self.h)


def replay_sample(seed: int, step: int, size: int, B: int) -> np.ndarray:
    idx = np.zeros(B, dtype=np.uint32)
    lib().orc_replay_sample(seed, step, size, B, _ptr(idx))
    return idx
