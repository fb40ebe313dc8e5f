"""The N > 1 path on CPU: world_size 2 over gloo.

Environments are independent, so a multi-GPU run shards the env range with no data-path collective: rank r simulates
envs [lo, hi) of the global batch with Philox keyed by the GLOBAL env id (SimParams.env_offset -> mig_params_t.env_base),
and the only communication is the reduction of the timing (max over ranks) and of the event count (sum) that bench.py
reports.  There is no GPU here, so the per-env compute stands in as the oracle called with the same global ids the CUDA
path would use (tests may use the oracle); what is tested is the host logic: the partition, the id offsets, the
placement invariance of the results and the reduction helper bench.py calls.
"""
import dataclasses
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle as O
from paper_2606_25082_b200 import workloads as W

N_ENVS = 10


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = W.config_c3(N_ENVS)
    lo, hi = W.shard_range(N_ENVS, rank, world)
    sp = dataclasses.replace(wl.params, env_offset=lo)               # what bench.py / a multi-GPU user passes to MigSim
    hashes, events = [], 0
    for e in range(hi - lo):                                         # local env index, as in the rank's own arrays
        r = O.rollout(sp, wl.seed, e + sp.env_offset, algo=int(wl.algo[lo + e]), cfg0=int(wl.cfg0[lo + e]), policy=wl.policy,
                      table=wl.table[lo + e])
        hashes.append(int(r.totals["trace_hash"]))
        events += int(r.totals["n_jobs"] + r.totals["n_completed"])
    seconds = 1.0 + rank                                             # rank 1 is the slow one
    t_max, ev_sum = W.reduce_over_ranks(seconds, events)
    gathered = [None] * world
    dist.all_gather_object(gathered, (lo, hi, hashes, events))
    if rank == 0:
        np.save(os.path.join(out_dir, "hashes.npy"), np.array([h for g in gathered for h in g[2]], dtype=np.uint64))
        np.save(os.path.join(out_dir, "meta.npy"), np.array([t_max, ev_sum, sum(g[3] for g in gathered)] + [x for g in gathered for x in g[:2]], dtype=np.float64))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_ranges_partition_the_batch():
    for n in (1, 7, 10, 65536):
        for world in (1, 2, 3, 8):
            rs = [W.shard_range(n, r, world) for r in range(world)]
            assert rs[0][0] == 0 and rs[-1][1] == n
            assert all(rs[i][1] == rs[i + 1][0] for i in range(world - 1))
            assert max(hi - lo for lo, hi in rs) - min(hi - lo for lo, hi in rs) <= 1


def test_reduce_over_ranks_is_identity_without_a_process_group():
    assert W.reduce_over_ranks(1.5, 7) == (1.5, 7)


@pytest.mark.timeout(300)
def test_world_size_2_gloo_sharding_is_placement_invariant(tmp_path):
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    hashes = np.load(tmp_path / "hashes.npy")
    meta = np.load(tmp_path / "meta.npy")
    # one process over the whole batch gives the same days
    wl = W.config_c3(N_ENVS)
    ref, ev_ref = [], 0
    for e in range(N_ENVS):
        r = O.rollout(wl.params, wl.seed, e, algo=int(wl.algo[e]), cfg0=int(wl.cfg0[e]), policy=wl.policy, table=wl.table[e])
        ref.append(int(r.totals["trace_hash"]))
        ev_ref += int(r.totals["n_jobs"] + r.totals["n_completed"])
    assert hashes.tolist() == ref and len(set(ref)) == N_ENVS
    assert meta[0] == 2.0                                            # max over ranks of the time
    assert int(meta[1]) == ev_ref == int(meta[2])                    # sum over ranks of the units
    assert meta[3:].tolist() == [0, 5, 5, 10]
