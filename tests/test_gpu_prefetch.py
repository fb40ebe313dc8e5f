"""mig_sim_set_prefetch (the next episode's arrival lists drawn in the tail of a full-day launch): the days
are the same with the setting on or off -- records, totals and trace hashes byte for byte -- whatever the call sequence
(consecutive episodes, an episode that was not drawn ahead, steps in between, a batch whose last warp is partial, BASELINE
C5 at full size in the launch configuration bench.py times), and a sample of them is checked against the oracle directly.
"""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _workload(n_envs):
    """The C5 recipe (heavy load, hourly TABLE policy, queues that spill into the global ring) on a smaller batch."""
    return W.CONFIGS["C5"](n_envs)


def _days(B, wl, n, episodes, prefetch, steps_before=()):
    sim = B.MigSim(wl.params, n, wl.seed)
    sim.set_envs_per_warp(32)                       # the tail draws only in launches with 32 environments per warp
    if prefetch:
        sim.set_prefetch(True)
        assert sim.get_prefetch()
    d_algo, d_cfg0, d_table = dev(wl.algo[:n]), dev(wl.cfg0[:n]), dev(wl.table[:n])
    out = []
    for ep in episodes:
        recs, tot = sim.alloc_recs(), sim.alloc_totals()
        sim.reset(ep, d_algo, d_cfg0)
        if ep in steps_before:                      # a day that starts with explicit steps: not a full-day launch
            act = dev(np.full(n, 1, np.uint8))
            for _ in range(3):
                sim.step(act)
        sim.rollout(wl.policy, table=d_table, recs_out=recs, totals_out=tot)
        torch.cuda.synchronize()
        out.append((B.recs_to_numpy(recs).tobytes(), B.totals_to_numpy(tot).copy()))
    return out


@pytest.mark.parametrize("n,mixed", [(2048, False), (1000, False), (512, True)], ids=["2048", "1000", "512-all-algorithms"])
def test_prefetch_days_are_identical(n, mixed):
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_25082_b200 import binding as B
    wl = _workload(n)
    if mixed:                                       # EDF-FS, EDF-SS, LLF, LALF and restricted EDF-SS side by side: the kernel's generic body
        wl.algo[:] = np.arange(n, dtype=np.uint8) % 5
    # 0, 1, 2: each drawn ahead by the one before; 7: not drawn ahead (what was drawn for 3 is dropped); 8: ahead again;
    # 8 once more: the lists drawn for 9 stay unused; 9 begins with three explicit steps (no full-day launch) and 10 follows
    episodes = [0, 1, 2, 7, 8, 8, 9, 10]
    on = _days(B, wl, n, episodes, True, steps_before=(9,))
    off = _days(B, wl, n, episodes, False, steps_before=(9,))
    for ep, a, b in zip(episodes, on, off):
        assert a[0] == b[0], "records of episode %d differ with prefetch on" % ep
        assert a[1].tobytes() == b[1].tobytes(), "totals of episode %d differ with prefetch on" % ep
    # the oracle on a sample of the days that WERE drawn ahead (episodes 1 and 2)
    ph = O.ParamsHolder(wl.params)
    for k, ep in ((1, 1), (2, 2)):
        tot = on[k][1]
        for e in (0, 31, 32, n // 2 + 5, n - 1):
            r = O.rollout(ph, wl.seed, e, episode=ep, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy, table=wl.table[e])
            assert tot[e].tobytes() == r.totals.tobytes(), "episode %d env %d differs from the oracle" % (ep, e)


def test_prefetch_full_size_c5_in_the_bench_configuration():
    """BASELINE C5 at full size (65 536 env-days, 32 per warp by the library's own choice: the launch bench.py times): three
    consecutive episodes with drawing ahead on equal the same episodes with it off, every env; a sample against the oracle."""
    from paper_2606_25082_b200 import binding as B
    n = 65536
    wl = W.CONFIGS["C5"](n)
    d_algo, d_cfg0, d_table = dev(wl.algo), dev(wl.cfg0), dev(wl.table)
    res = {}
    for on in (True, False):
        sim = B.MigSim(wl.params, n, wl.seed)
        if on:
            sim.set_prefetch(True)
        out = []
        for ep in (0, 1, 2):
            recs, tot = sim.alloc_recs(), sim.alloc_totals()
            sim.reset(ep, d_algo, d_cfg0)
            sim.rollout(wl.policy, table=d_table, recs_out=recs, totals_out=tot)
            torch.cuda.synchronize()
            out.append((recs.cpu(), B.totals_to_numpy(tot).copy()))
            del recs, tot
        res[on] = out
        sim.close()
        del sim
        torch.cuda.empty_cache()
    for ep in (0, 1, 2):
        assert torch.equal(res[True][ep][0], res[False][ep][0]), "records of episode %d differ" % ep
        assert res[True][ep][1].tobytes() == res[False][ep][1].tobytes(), "totals of episode %d differ" % ep
    ph = O.ParamsHolder(wl.params)
    for e in (0, 4095, 32768, 65535):
        r = O.rollout(ph, wl.seed, e, episode=2, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy, table=wl.table[e])
        assert res[True][2][1][e].tobytes() == r.totals.tobytes(), "episode 2 env %d differs from the oracle" % e


def test_prefetch_needs_lists_and_survives_a_new_capacity():
    from paper_2606_25082_b200 import binding as B
    wl = _workload(256)
    n = 256
    sim = B.MigSim(wl.params, n, wl.seed)
    sim.set_envs_per_warp(32)
    sim.set_prefetch(True)
    d_algo, d_cfg0, d_table = dev(wl.algo[:n]), dev(wl.cfg0[:n]), dev(wl.table[:n])
    ref = None
    for cap in (0xFFFFFFFF, 512, 0xFFFFFFFF):       # a new capacity drops what was drawn ahead; small lists are continued inline
        sim.set_arrival_buffer(cap)
        assert sim.get_prefetch()
        tots = []
        for ep in (3, 4):
            tot = sim.alloc_totals()
            sim.reset(ep, d_algo, d_cfg0)
            sim.rollout(wl.policy, table=d_table, totals_out=tot)
            torch.cuda.synchronize()
            tots.append(B.totals_to_numpy(tot).tobytes())
        if ref is None:
            ref = tots
        assert tots == ref
    sim.set_arrival_buffer(0)                        # no lists: nothing to draw ahead into
    with pytest.raises(Exception):
        sim.set_prefetch(False); sim.set_prefetch(True)
