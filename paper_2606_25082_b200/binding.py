"""Thin ctypes binding of libmigsim.so (include/migsim.h): same names, argument marshalling only.

PyTorch is used for device memory and streams; every step of the simulated path runs in the CUDA kernels.
There is no CPU fallback: if the library cannot be loaded, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C

import numpy as np
import torch

from . import _build
from .workloads import STATE_DIM, QNetWeights, SimParams

MIG_OK, MIG_EINVAL, MIG_ENOMEM, MIG_ECUDA, MIG_ESTATE = 0, -1, -2, -3, -4
POLICY_STATIC, POLICY_TABLE, POLICY_DQN, POLICY_BINNED = 0, 1, 2, 3

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
JOB_DTYPE = np.dtype([("arr", "<i4"), ("cls", "<u4"), ("dur7", "<i4"), ("due", "<i4")])
assert EVENT_DTYPE.itemsize == 16 and REC_DTYPE.itemsize == 64 and TOTALS_DTYPE.itemsize == 80

EXPORTS = (
    "mig_last_error", "mig_version", "mig_sim_create", "mig_sim_destroy", "mig_sim_reset", "mig_sim_step",
    "mig_sim_rollout", "mig_sim_totals", "mig_sim_rollout_host", "mig_qnet_create", "mig_qnet_destroy", "mig_q_eval",
    "mig_sim_debug_trace", "mig_sim_debug_set_jobs", "mig_debug_div_magic", "mig_sim_launch_count", "mig_sim_set_tile",
    "mig_sim_get_tile", "mig_sim_set_arrival_buffer", "mig_sim_get_arrival_buffer", "mig_sim_set_envs_per_warp",
    "mig_sim_kernel_name", "mig_sim_set_profiling", "mig_sim_kernel_times", "mig_sim_aux", "mig_et_reduce",
    "mig_dqn_create", "mig_dqn_destroy", "mig_replay_push", "mig_replay_size", "mig_dqn_train_step", "mig_dqn_train_on",
    "mig_dqn_sync_target", "mig_dqn_q", "mig_dqn_get_weights", "mig_dqn_launch_count", "mig_q_forward_static",
    "mig_sim_set_prefetch", "mig_sim_get_prefetch")


class MigError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("migsim error %d: %s" % (code, msg))
        self.code = code


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
        ("w_energy", C.c_float), ("w_tardy", C.c_float), ("env_base", C.c_uint32), ("decide_on_events", C.c_uint32),
        ("speed_nomig", C.c_void_p), ("p_idle_nomig_mw", C.c_int32), ("p_busy_nomig_mw", C.c_int32),
        ("repart_all_down", C.c_uint32), ("gamma", C.c_float),
        ("n_tbins", C.c_uint32), ("n_dbins", C.c_uint32), ("n_abins", C.c_uint32),
        ("dbin_edges", C.c_void_p), ("abin_edges", C.c_void_p), ("util_hist", C.c_uint32),
    ]


_lib = None


def lib():
    """Loads (building it first if the source is newer) libmigsim.so.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, u32, u64, i32, f32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int, C.c_float
        L.mig_last_error.restype = C.c_char_p
        L.mig_version.restype = C.c_char_p
        L.mig_sim_create.argtypes = [C.POINTER(vp), C.POINTER(_Params), u32, u64]
        L.mig_sim_destroy.argtypes = [vp]
        L.mig_sim_reset.argtypes = [vp, u32, vp, vp, vp, vp]
        L.mig_sim_step.argtypes = [vp] * 9
        L.mig_sim_rollout.argtypes = [vp, i32, vp, vp, f32, vp, vp, vp]
        L.mig_sim_totals.argtypes = [vp, vp, vp]
        L.mig_sim_rollout_host.argtypes = [vp, u32, vp, vp, i32, vp, vp, f32, vp, vp]
        L.mig_qnet_create.argtypes = [C.POINTER(vp), vp, vp, vp, vp, vp, vp, u32, u32]
        L.mig_qnet_destroy.argtypes = [vp]
        L.mig_q_eval.argtypes = [vp, vp, u32, vp, vp, vp]
        L.mig_sim_debug_trace.argtypes = [vp, u32, i32, vp, vp, vp, u32, vp, vp, vp]
        L.mig_sim_debug_set_jobs.argtypes = [vp, vp, u32]
        L.mig_debug_div_magic.argtypes = [u32, C.POINTER(u32), C.POINTER(u32)]
        L.mig_sim_launch_count.argtypes = [vp]
        L.mig_sim_launch_count.restype = u64
        L.mig_sim_set_tile.argtypes = [vp, i32]
        L.mig_sim_get_tile.argtypes = [vp]
        L.mig_sim_set_arrival_buffer.argtypes = [vp, C.c_uint32]
        L.mig_sim_set_envs_per_warp.argtypes = [vp, C.c_uint32]
        L.mig_sim_set_prefetch.argtypes = [vp, i32]
        L.mig_sim_get_prefetch.argtypes = [vp]
        L.mig_sim_kernel_name.argtypes = [vp]
        L.mig_sim_kernel_name.restype = C.c_char_p
        L.mig_sim_set_profiling.argtypes = [vp, i32]
        L.mig_sim_kernel_times.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(C.c_uint32)]
        L.mig_sim_get_arrival_buffer.argtypes = [vp]
        L.mig_sim_get_arrival_buffer.restype = C.c_uint32
        L.mig_sim_aux.argtypes = [vp, vp, vp, vp]
        L.mig_et_reduce.argtypes = [vp, vp, vp, u32, u32, vp, vp]
        L.mig_dqn_create.argtypes = [C.POINTER(vp), vp, vp, vp, vp, vp, vp, u32, u32, u32, u32, f32, f32, u64]
        L.mig_dqn_destroy.argtypes = [vp]
        L.mig_replay_push.argtypes = [vp, vp, vp, vp, vp, vp, u32, vp]
        L.mig_replay_size.argtypes = [vp]
        L.mig_replay_size.restype = u32
        L.mig_dqn_train_step.argtypes = [vp, u32, vp, vp]
        L.mig_dqn_train_on.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
        L.mig_dqn_sync_target.argtypes = [vp, vp]
        L.mig_dqn_q.argtypes = [vp, i32, vp, u32, vp, vp]
        L.mig_dqn_get_weights.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
        L.mig_q_forward_static.argtypes = [vp, vp, vp, vp, vp, vp, u32, u32, vp, u32, vp, vp]
        L.mig_dqn_launch_count.argtypes = [vp]
        L.mig_dqn_launch_count.restype = u64
        _lib = L
    return _lib


def _check(rc):
    if rc != MIG_OK:
        raise MigError(rc, lib().mig_last_error().decode())


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t, dtype=None, numel=None):
    """Device pointer of a torch tensor (argument marshalling: must be CUDA, contiguous)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError("expected dtype %s, got %s" % (dtype, t.dtype))
    if numel is not None and t.numel() * t.element_size() < numel:
        raise ValueError("tensor too small: %d bytes < %d" % (t.numel() * t.element_size(), numel))
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def div_magic(v: int):
    m, sh = C.c_uint32(), C.c_uint32()
    _check(lib().mig_debug_div_magic(v, C.byref(m), C.byref(sh)))
    return m.value, sh.value


def _fill_params(sp: SimParams) -> tuple[_Params, tuple]:
    sp = sp.normalised()
    s = _Params()
    s.n_classes, s.n_configs = sp.n_classes, sp.n_configs
    keep = (sp.speed, sp.dur7_q, sp.class_cum, sp.slack_q10, sp.size_at_slot, sp.accept_thr)
    s.speed, s.dur7_q, s.class_cum = _hp(sp.speed), _hp(sp.dur7_q), _hp(sp.class_cum)
    s.slack_q10, s.size_at_slot, s.accept_thr = _hp(sp.slack_q10), _hp(sp.size_at_slot), _hp(sp.accept_thr)
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
    s.w_energy, s.w_tardy, s.env_base = sp.w_energy, sp.w_tardy, sp.env_offset
    s.decide_on_events = int(sp.decide_on_events)
    keep = keep + (sp.speed_nomig, sp.dbin_edges, sp.abin_edges)
    s.speed_nomig = _hp(sp.speed_nomig)
    s.p_idle_nomig_mw, s.p_busy_nomig_mw = int(sp.p_idle_nomig_mw), int(sp.p_busy_nomig_mw)
    s.repart_all_down, s.gamma = int(sp.repart_all_down), float(sp.gamma)
    s.n_tbins, s.n_dbins, s.n_abins = int(sp.n_tbins), int(sp.n_dbins), int(sp.n_abins)
    s.dbin_edges, s.abin_edges = _hp(sp.dbin_edges), _hp(sp.abin_edges)
    s.util_hist = int(sp.util_hist)
    return s, keep


class QNet:
    """mig_qnet_create / mig_q_eval / mig_qnet_destroy."""

    def __init__(self, qw: QNetWeights):
        arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (qw.W1, qw.b1, qw.W2, qw.b2, qw.W3, qw.b3)]
        self.hidden, self.n_actions = int(arrs[0].shape[1]), int(arrs[4].shape[1])
        self.h = C.c_void_p()
        _check(lib().mig_qnet_create(C.byref(self.h), *[_hp(a) for a in arrs], self.hidden, self.n_actions))

    def q_eval(self, state: torch.Tensor, q_out: torch.Tensor | None = None, argmax_out: torch.Tensor | None = None,
               stream=None):
        B = state.numel() // STATE_DIM
        _check(lib().mig_q_eval(self.h, _dp(state, torch.float32), B, _dp(q_out, torch.float32, B * self.n_actions * 4),
                                _dp(argmax_out, torch.uint8, B), _stream(stream)))

    def close(self):
        if getattr(self, "h", None) and _lib is not None:      # (at interpreter shutdown the module may be gone already)
            _lib.mig_qnet_destroy(self.h)
        self.h = None

    __del__ = close


class Dqn:
    """mig_dqn_* / mig_replay_*: DQN training on the tensor cores (online + frozen target network, replay ring on the device)."""

    def __init__(self, qw: QNetWeights, replay_capacity: int, batch: int, gamma: float, lr: float, seed: int):
        if not torch.cuda.is_available():
            raise MigError(MIG_ECUDA, "no CUDA device: the training step has no CPU fallback")
        arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (qw.W1, qw.b1, qw.W2, qw.b2, qw.W3, qw.b3)]
        self.hidden, self.n_actions, self.batch = int(arrs[0].shape[1]), int(arrs[4].shape[1]), int(batch)
        self.h = C.c_void_p()
        _check(lib().mig_dqn_create(C.byref(self.h), *[_hp(a) for a in arrs], self.hidden, self.n_actions, int(replay_capacity),
                                    self.batch, float(gamma), float(lr), int(seed)))

    def close(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.mig_dqn_destroy(self.h)
        self.h = None

    __del__ = close

    def push(self, s, a, r, s2, done=None, stream=None):
        n = a.numel()
        _check(lib().mig_replay_push(self.h, _dp(s, torch.float32, n * STATE_DIM * 4), _dp(a, torch.uint8, n), _dp(r, torch.float32, n * 4),
                                     _dp(s2, torch.float32, n * STATE_DIM * 4), _dp(done, torch.uint8, n), n, _stream(stream)))

    def replay_size(self) -> int:
        return int(lib().mig_replay_size(self.h))

    def train_step(self, step: int, loss_out=None, stream=None):
        _check(lib().mig_dqn_train_step(self.h, int(step), _dp(loss_out, torch.float32, 4), _stream(stream)))

    def train_on(self, s, a, r, s2, done=None, loss_out=None, stream=None):
        B = self.batch
        _check(lib().mig_dqn_train_on(self.h, _dp(s, torch.float32, B * STATE_DIM * 4), _dp(a, torch.uint8, B), _dp(r, torch.float32, B * 4),
                                      _dp(s2, torch.float32, B * STATE_DIM * 4), _dp(done, torch.uint8, B), _dp(loss_out, torch.float32, 4),
                                      _stream(stream)))

    def sync_target(self, stream=None):
        _check(lib().mig_dqn_sync_target(self.h, _stream(stream)))

    def q(self, state: torch.Tensor, which: int = 0, q_out=None, stream=None):
        n = state.numel() // STATE_DIM
        q_out = torch.empty((n, self.n_actions), dtype=torch.float32, device="cuda") if q_out is None else q_out
        _check(lib().mig_dqn_q(self.h, int(which), _dp(state, torch.float32), n, _dp(q_out, torch.float32, n * self.n_actions * 4), _stream(stream)))
        return q_out

    def weights(self, which: int = 0) -> QNetWeights:
        H, A = self.hidden, self.n_actions
        arrs = [np.zeros(sh, dtype=np.float32) for sh in ((STATE_DIM, H), (H,), (H, H), (H,), (H, A), (A,))]
        _check(lib().mig_dqn_get_weights(self.h, int(which), *[_hp(a) for a in arrs]))
        return QNetWeights(*arrs)

    def launch_count(self) -> int:
        return int(lib().mig_dqn_launch_count(self.h))


# lanes per environment passed to mig_sim_set_tile by MigSim() when its `tile` argument is 0 (0 = the library's choice)
DEFAULT_TILE = 0


class MigSim:
    """mig_sim_* calls on one handle.  Tensors are caller-owned CUDA tensors; nothing is allocated here except by
    the convenience helpers whose names start with ``alloc_``."""

    def __init__(self, sp: SimParams, n_envs: int, seed: int, tile: int = 0):
        if not torch.cuda.is_available():
            raise MigError(MIG_ECUDA, "no CUDA device: the simulator has no CPU fallback")
        self.sp, self.n_envs, self.seed = sp, int(n_envs), int(seed)
        self.n_epochs = sp.n_epochs
        ps, keep = _fill_params(sp)
        self.h = C.c_void_p()
        _check(lib().mig_sim_create(C.byref(self.h), C.byref(ps), self.n_envs, self.seed))
        tile = tile or DEFAULT_TILE
        if tile:
            self.set_tile(tile)

    def set_tile(self, lanes_per_env: int):
        _check(lib().mig_sim_set_tile(self.h, int(lanes_per_env)))

    def get_tile(self) -> int:
        return int(lib().mig_sim_get_tile(self.h))

    def set_envs_per_warp(self, envs_per_warp: int):
        _check(lib().mig_sim_set_envs_per_warp(self.h, int(envs_per_warp)))

    def set_arrival_buffer(self, entries_per_env: int):
        _check(lib().mig_sim_set_arrival_buffer(self.h, int(entries_per_env)))

    def get_arrival_buffer(self) -> int:
        return int(lib().mig_sim_get_arrival_buffer(self.h))

    def set_prefetch(self, on: bool):
        _check(lib().mig_sim_set_prefetch(self.h, 1 if on else 0))

    def get_prefetch(self) -> bool:
        return bool(lib().mig_sim_get_prefetch(self.h))

    def close(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.mig_sim_destroy(self.h)
        self.h = None

    __del__ = close

    # ---- allocation helpers (plain torch) -------------------------------------------------------------------------
    def alloc_recs(self):
        return torch.zeros((self.n_epochs + 1, self.n_envs, 64), dtype=torch.uint8, device="cuda")

    def alloc_totals(self):
        return torch.zeros((self.n_envs, 80), dtype=torch.uint8, device="cuda")

    def alloc_state(self):
        return torch.zeros((self.n_envs, STATE_DIM), dtype=torch.float32, device="cuda")

    # ---- the C ABI -------------------------------------------------------------------------------------------------
    def reset(self, episode: int, algo: torch.Tensor, cfg0: torch.Tensor, state_out=None, stream=None):
        _check(lib().mig_sim_reset(self.h, episode, _dp(algo, torch.uint8, self.n_envs), _dp(cfg0, torch.uint8, self.n_envs),
                                   _dp(state_out, torch.float32, self.n_envs * STATE_DIM * 4), _stream(stream)))

    def step(self, action: torch.Tensor, state_out=None, reward_out=None, energy_out=None, tard_out=None, rec_out=None,
             drain_rec_out=None, stream=None):
        n = self.n_envs
        _check(lib().mig_sim_step(self.h, _dp(action, torch.uint8, n), _dp(state_out, torch.float32, n * STATE_DIM * 4),
                                  _dp(reward_out, torch.float32, n * 4), _dp(energy_out, torch.int64, n * 8),
                                  _dp(tard_out, torch.int64, n * 8), _dp(rec_out, torch.uint8, n * 64),
                                  _dp(drain_rec_out, torch.uint8, n * 64), _stream(stream)))

    def rollout(self, policy: int, table=None, qnet: QNet | None = None, epsilon: float = 0.0, recs_out=None,
                totals_out=None, stream=None):
        n = self.n_envs
        tb = self.sp.n_configs * self.sp.n_tbins * self.sp.binned_codes ** 3 if policy == POLICY_BINNED else n * self.n_epochs * 4
        _check(lib().mig_sim_rollout(self.h, policy, _dp(table, torch.uint8, tb),
                                     qnet.h if qnet is not None else None, float(epsilon),
                                     _dp(recs_out, torch.uint8, (self.n_epochs + 1) * n * 64),
                                     _dp(totals_out, torch.uint8, n * 80), _stream(stream)))

    def aux(self, return_out=None, util_s_out=None, stream=None):
        """mig_sim_aux: discounted return dev[n_envs] fp32 and / or seconds per utilisation level dev[n_envs][8] int32."""
        _check(lib().mig_sim_aux(self.h, _dp(return_out, torch.float32, self.n_envs * 4), _dp(util_s_out, torch.int32, self.n_envs * 32),
                                 _stream(stream)))

    def totals(self, totals_out, stream=None):
        _check(lib().mig_sim_totals(self.h, _dp(totals_out, torch.uint8, self.n_envs * 80), _stream(stream)))

    def rollout_host(self, episode: int, algo: np.ndarray, cfg0: np.ndarray, policy: int, table: np.ndarray | None,
                     qnet: QNet | None, epsilon: float, recs_out: np.ndarray | None, totals_out: np.ndarray):
        """HOST buffers in, HOST buffers out (the e2e path of bench.py)."""
        n = self.n_envs
        assert algo.dtype == np.uint8 and cfg0.dtype == np.uint8 and algo.size == n and cfg0.size == n
        assert totals_out.dtype == TOTALS_DTYPE and totals_out.size == n and totals_out.flags.c_contiguous
        if recs_out is not None:
            assert recs_out.dtype == REC_DTYPE and recs_out.size == n * (self.n_epochs + 1) and recs_out.flags.c_contiguous
        if table is not None:
            want = self.sp.n_configs * self.sp.n_tbins * self.sp.binned_codes ** 3 if policy == POLICY_BINNED else n * self.n_epochs * 4
            assert table.dtype == np.uint8 and table.size == want and table.flags.c_contiguous
        _check(lib().mig_sim_rollout_host(self.h, episode, _hp(algo), _hp(cfg0), policy, _hp(table),
                                          qnet.h if qnet is not None else None, float(epsilon), _hp(recs_out), _hp(totals_out)))

    def debug_trace(self, env: int, policy: int = POLICY_STATIC, table=None, actions=None, cap_events: int = 1 << 20,
                    stream=None):
        """Returns (events ndarray[EVENT_DTYPE], totals record) of one env re-run from the last reset."""
        buf = torch.zeros((cap_events, 16), dtype=torch.uint8, device="cuda")
        n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
        tot = torch.zeros((1, 80), dtype=torch.uint8, device="cuda")
        _check(lib().mig_sim_debug_trace(self.h, env, policy, _dp(table, torch.uint8), _dp(actions, torch.uint8, self.n_epochs),
                                         _dp(buf), cap_events, _dp(n_out), _dp(tot), _stream(stream)))
        torch.cuda.synchronize()
        n = int(n_out.item())
        if n > cap_events:
            raise ValueError("trace buffer too small: %d events" % n)
        ev = buf[:n].cpu().numpy().view(EVENT_DTYPE).reshape(-1)
        return ev, tot.cpu().numpy().view(TOTALS_DTYPE).reshape(-1)[0]

    def debug_set_jobs(self, jobs: np.ndarray | None):
        if jobs is None or len(jobs) == 0:
            _check(lib().mig_sim_debug_set_jobs(self.h, None, 0))
            return
        j = np.ascontiguousarray(jobs, dtype=JOB_DTYPE)
        _check(lib().mig_sim_debug_set_jobs(self.h, _hp(j), len(j)))

    def launch_count(self) -> int:
        return int(lib().mig_sim_launch_count(self.h))

    def kernel_name(self) -> str:
        return lib().mig_sim_kernel_name(self.h).decode()

    def set_profiling(self, on: bool):
        _check(lib().mig_sim_set_profiling(self.h, int(bool(on))))

    def kernel_times(self):
        """({"gen": ms, "sim": ms, "qnet": ms}, {... launches}) since the last call (needs set_profiling(True))."""
        ms, n = (C.c_float * 3)(), (C.c_uint32 * 3)()
        _check(lib().mig_sim_kernel_times(self.h, ms, n))
        names = ("gen", "sim", "qnet")
        return {k: float(ms[i]) for i, k in enumerate(names)}, {k: int(n[i]) for i, k in enumerate(names)}


def recs_to_numpy(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(REC_DTYPE).reshape(t.shape[:-1])


def totals_to_numpy(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().view(TOTALS_DTYPE).reshape(t.shape[:-1])


Q_STATIC_MAX_ROWS = 2048                                     # MIG_Q_STATIC_MAX_ROWS of include/migsim.h


def q_forward_static(W1, b1, W2, b2, W3, b3, state: torch.Tensor, q_out: torch.Tensor, stream=None):
    """mig_q_forward_static: Q-values on the tensor cores with no allocation anywhere (the scratch is a static array of the
    library; at most Q_STATIC_MAX_ROWS rows per call).  All arguments are caller-owned CUDA tensors: weights in
    mig_qnet_create's layout, state [n][64], q_out [n][n_actions].  Calls that overlap on the GPU race on the scratch."""
    H, A = int(W2.shape[0]), int(W3.shape[1])
    n = state.numel() // STATE_DIM
    _check(lib().mig_q_forward_static(_dp(W1, torch.float32, STATE_DIM * H * 4), _dp(b1, torch.float32, H * 4), _dp(W2, torch.float32, H * H * 4),
                                      _dp(b2, torch.float32, H * 4), _dp(W3, torch.float32, H * A * 4), _dp(b3, torch.float32, A * 4), H, A,
                                      _dp(state, torch.float32), n, _dp(q_out, torch.float32, n * A * 4), _stream(stream)))
    return q_out


def et_reduce(x, y, group, n_groups: int):
    """mig_et_reduce: ET per group and the global scaling factor a; host arrays."""
    x = np.ascontiguousarray(x, dtype=np.float64); y = np.ascontiguousarray(y, dtype=np.float64)
    g = np.ascontiguousarray(group, dtype=np.uint32)
    et = np.zeros(n_groups, dtype=np.float64)
    a = C.c_double()
    _check(lib().mig_et_reduce(_hp(x), _hp(y), _hp(g), len(x), n_groups, _hp(et), C.byref(a)))
    return et, a.value
