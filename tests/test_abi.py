"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/migsim.h declares, validates its
parameter tables, computes exact division constants, and FAILS LOUDLY without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

from paper_2606_25082_b200 import binding as B
from paper_2606_25082_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "migsim.h")).read()
    declared = set(re.findall(r"\b(mig_[a-z0-9_]+)\s*\(", hdr))
    declared -= {"mig_params_t", "mig_sim_t"}
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    L = B.lib()
    for name in declared:
        assert getattr(L, name) is not None
    assert b"sm_100a" in L.mig_version()


def test_struct_layouts_match_header_sizes():
    assert B.REC_DTYPE.itemsize == 64 and B.TOTALS_DTYPE.itemsize == 80 and B.EVENT_DTYPE.itemsize == 16 and B.JOB_DTYPE.itemsize == 16


def test_div_magic_is_exact():
    rng = np.random.default_rng(0)
    vs = list(range(1, 300)) + [317, 449, 550, 635, 840, 65535, 65536, 65537, (1 << 24) - 1, 1 << 24] + \
        [int(x) for x in rng.integers(1, 1 << 24, size=300)]
    edge = np.array([0, 1, 2, 3, (1 << 31) - 1, (1 << 31) - 2, 1 << 30, (1 << 30) - 1], dtype=np.uint64)
    for v in vs:
        m, sh = B.div_magic(v)
        xs = np.concatenate([edge, rng.integers(0, 1 << 31, size=2000).astype(np.uint64),
                             (np.arange(1, 200, dtype=np.uint64) * np.uint64(v)) % np.uint64(1 << 31),
                             ((np.arange(1, 200, dtype=np.uint64) * np.uint64(v)) - np.uint64(1)) % np.uint64(1 << 31)])
        if v == 1:
            assert sh == 32
            continue
        q = ((xs * np.uint64(m)) >> np.uint64(32)) >> np.uint64(sh)
        assert np.array_equal(q, xs // np.uint64(v)), v
    with pytest.raises(B.MigError):
        B.div_magic(0)


def _create(sp, n_envs=4):
    ps, keep = B._fill_params(sp)
    h = C.c_void_p()
    rc = B.lib().mig_sim_create(C.byref(h), C.byref(ps), n_envs, 1)
    msg = B.lib().mig_last_error().decode()
    if rc == 0:
        B.lib().mig_sim_destroy(h)
    return rc, msg


def test_create_validates_tables_before_touching_the_device():
    base = W.config_c2(4).params
    import dataclasses

    def with_(**kw):
        return dataclasses.replace(base, **kw)

    bad_size = base.size_at_slot.copy(); bad_size[0, 0] = 5
    overlap = base.size_at_slot.copy(); overlap[1] = [4, 0, 3, 0, 0, 0, 0]
    beyond = base.size_at_slot.copy(); beyond[1] = [0, 0, 0, 0, 0, 4, 0]
    zero_speed = base.speed.copy(); zero_speed[2, 1] = 0
    nonmono = base.dur7_q.copy(); nonmono[0, 10] = nonmono[0, 9] - 1
    cum = base.class_cum.copy(); cum[-1] = 5
    cases = [
        (with_(size_at_slot=bad_size), "not in {1,2,3,4,7}"),
        (with_(size_at_slot=overlap), "overlap"),
        (with_(size_at_slot=beyond), "exceeds 7 slots"),
        (with_(speed=zero_speed), "speed"),
        (with_(dur7_q=nonmono), "non-decreasing"),
        (with_(class_cum=cum), "class_cum"),
        (with_(cap=0), "cap"), (with_(cap=2048), "cap"),
        (with_(crit_max=16), "crit_max"),
        (with_(t_limit_s=86400), "t_limit_s"),
        (with_(day_s=90000), "day_s"),
    ]
    for sp, frag in cases:
        rc, msg = _create(sp)
        assert rc == B.MIG_EINVAL and frag in msg, (rc, msg, frag)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback_without_a_device():
    rc, msg = _create(W.config_c2(4).params)
    assert rc == B.MIG_ECUDA and "no CPU fallback" in msg
    with pytest.raises(B.MigError):
        B.MigSim(W.config_c2(4).params, 4, 1)
    with pytest.raises(B.MigError):
        B.QNet(W.make_qnet(0))
