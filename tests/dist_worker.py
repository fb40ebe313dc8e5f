"""Worker of tests/test_gpu_multiproc.py: rank r of a torch.distributed job simulates envs [r n, (r + 1) n) of a global batch on
cuda:0 (every rank on the SAME GPU: this run has one) exactly as bench.py does for N > 1 -- env_offset = rank * n, Philox keyed
by the global env id -- and rank 0 checks the gathered totals against ONE handle of world * n envs.  gloo carries the gather
(NCCL refuses two ranks on one device); the NCCL path itself is exercised by bench.py under BENCH_FORCE_DIST=1."""
import dataclasses
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2606_25082_b200 import binding as B          # noqa: E402
from paper_2606_25082_b200 import workloads as W        # noqa: E402


def day(sp, n, seed, wl, lo):
    sim = B.MigSim(sp, n, seed)
    tot = sim.alloc_totals()
    sim.reset(0, torch.from_numpy(wl.algo[lo:lo + n].copy()).cuda(), torch.from_numpy(wl.cfg0[lo:lo + n].copy()).cuda())
    sim.rollout(wl.policy, table=torch.from_numpy(wl.table[lo:lo + n].copy()).cuda(), totals_out=tot)
    torch.cuda.synchronize()
    out = tot.cpu()
    sim.close()
    return out


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    n = 192
    wl = W.config_c3(world * n)
    lo, hi = W.shard_range(world * n, rank, world)
    assert (lo, hi) == (rank * n, (rank + 1) * n)
    mine = day(dataclasses.replace(wl.params, env_offset=rank * n), n, wl.seed, wl, lo)
    gathered = [torch.zeros_like(mine) for _ in range(world)] if rank == 0 else None
    dist.gather(mine, gathered, dst=0)
    ev = int(mine.numpy().view(B.TOTALS_DTYPE)["n_jobs"].sum())
    t, total = W.reduce_over_ranks(1.0 + rank, ev, device="cpu")
    if rank == 0:
        whole = day(wl.params, world * n, wl.seed, wl, 0)
        got = torch.cat(gathered, 0)
        assert torch.equal(got, whole), "sharded totals differ from the single handle"
        assert t == float(world) and total == int(whole.numpy().view(B.TOTALS_DTYPE)["n_jobs"].sum())
        print("DIST_OK world=%d envs=%d job-events=%d" % (world, world * n, total))
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
