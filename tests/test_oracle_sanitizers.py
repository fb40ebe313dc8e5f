"""Opt-in: the oracle's own tests re-run with oracle/mig_oracle.c built under AddressSanitizer + UndefinedBehaviorSanitizer.

    MIG_SANITIZE=1 python -m pytest tests/test_oracle_sanitizers.py -m sanitize

The oracle is the yardstick of every parity claim, so an out-of-bounds read or a signed overflow in it would make the
yardstick itself undefined.  (compute-sanitizer is closed on the GPU pool; the CUDA path's memory safety rests on the
bit-exact differential tests.)  Skipped by default: it roughly doubles the CPU suite.
"""
import glob
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
ORACLE_TESTS = ["tests/test_oracle_handworked.py", "tests/test_oracle_invariants.py", "tests/test_oracle_generator.py",
                "tests/test_oracle_qnet.py", "tests/test_oracle_pins_r2.py", "tests/test_oracle_dqn.py", "tests/test_oracle_paper_form.py"]


def _runtime(name):
    out = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


@pytest.mark.sanitize
@pytest.mark.skipif(os.environ.get("MIG_SANITIZE") != "1", reason="opt-in: set MIG_SANITIZE=1")
def test_oracle_suite_is_clean_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc sanitizer runtimes not installed")
    lib = str(tmp_path / "libmigoracle_san.so")
    srcs = sorted(glob.glob(os.path.join(ROOT, "oracle", "*.c")))
    subprocess.run(["gcc", "-O1", "-g", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-mfma", "-fsanitize=address,undefined",
                    "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", *srcs, "-o", lib, "-lm"], check=True)
    env = dict(os.environ, MIG_ORACLE_LIB=lib, LD_PRELOAD=asan + ":" + ubsan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", MIG_SANITIZE="0")
    tests = [t for t in ORACLE_TESTS if os.path.exists(os.path.join(ROOT, t))]
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", *tests], cwd=ROOT, env=env, capture_output=True, text=True)
    assert r.returncode == 0, r.stdout[-4000:] + r.stderr[-4000:]
    assert " passed" in r.stdout
