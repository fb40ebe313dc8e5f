"""Build the CPU oracle (plain C, gcc) into oracle/libmigoracle.so.  Test infrastructure only."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mig_oracle.c")
SRCS = [SRC, os.path.join(HERE, "dqn_oracle.c")]
HDR = os.path.join(HERE, "mig_oracle.h")
LIB = os.path.join(HERE, "libmigoracle.so")

# -ffp-contract=off: only the explicit fmaf() calls fuse; -mfma makes fmaf() one instruction.
CFLAGS = ["-O2", "-std=c99", "-fPIC", "-shared", "-Wall", "-Wextra", "-ffp-contract=off", "-mfma"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max([os.path.getmtime(f) for f in SRCS] + [os.path.getmtime(HDR)])):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *CFLAGS, *SRCS, "-o", tmp, "-lm"], check=True, cwd=HERE)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
