"""The N > 1 path of bench.py on the one GPU this run has: (a) two torch.distributed ranks, both on cuda:0,
each simulating its env range with env_offset = rank * n -- rank 1's results must be envs [n, 2n) of a single 2n-env handle;
(b) bench.py under torchrun with a one-rank NCCL group, so that the NCCL init and reduce_over_ranks(device="cuda") execute."""
import json
import os
import subprocess
import sys

import pytest
import torch

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(nproc, port, script, *args, env=None):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc), "--master-addr", "127.0.0.1",
           "--master-port", str(port), script, *args]
    return subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, **(env or {})), capture_output=True, text=True, timeout=900)


def test_two_ranks_on_one_gpu_partition_the_env_range():
    assert torch.cuda.is_available()
    r = _torchrun(2, 29611, os.path.join("tests", "dist_worker.py"))
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "DIST_OK world=2 envs=384" in r.stdout


def test_bench_under_torchrun_with_a_one_rank_nccl_group():
    r = _torchrun(1, 29612, "bench.py", "--gpus", "1", "--workload", "C3", "--envs", "512", "--steps", "2", "--warmup", "3", "--no-cpu-baseline",
                  "--no-step-api", env={"BENCH_FORCE_DIST": "1"})
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    line = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 1 and line["config"]["dist"] == "nccl, world 1" and line["value"] > 0 and line["gpu_launches"] > 0
