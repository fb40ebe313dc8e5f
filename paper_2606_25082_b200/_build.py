"""Builds libmigsim.so (hand-written CUDA for sm_100a + the C ABI of include/migsim.h) in-tree with nvcc."""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmigsim.so")
SOURCES = ["migsim.cu", "dqn.cu"]


def _deps() -> list[str]:
    """Every source the library is compiled from: csrc/*.cu, *.cuh, *.h and the public header (a stale .so must never
    pass a parity test: binding.lib() rebuilds when any of these is newer than libmigsim.so)."""
    out = []
    for pat in ("*.cu", "*.cuh", "*.h"):
        out += glob.glob(os.path.join(CSRC, pat))
    out += glob.glob(os.path.join(HERE, "..", "include", "*.h"))
    return sorted(out)

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "-cudart", "shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    mt = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > mt for d in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *SOURCES, "-o", tmp]
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
