"""CPU-only (sanitizer substitutes): the oracle built with AddressSanitizer and
UndefinedBehaviorSanitizer (g++ -fsanitize=address,undefined -fno-sanitize-recover=all) runs its
own pins -- P-1 ... P-12, the golden hand cases and the guard-branch workloads of
tests/test_oracle_pins.py, plus the one-ulp sensitivity runs -- in a child process.  Any
out-of-bounds index into the grid / particle arrays, use of freed memory, signed overflow,
misaligned or null access or invalid shift inside oracle/pic_oracle.cpp aborts the child.

The child is a fresh interpreter because the ASan runtime has to be the first library a process
loads (LD_PRELOAD); leak detection is off (CPython itself "leaks" at exit)."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _runtime(name):
    out = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True)
    path = out.stdout.strip()
    return path if os.path.isabs(path) and os.path.exists(path) else None


def test_oracle_pins_under_asan_ubsan():
    import pytest
    asan = _runtime("libasan.so")
    if asan is None:
        pytest.skip("no libasan.so next to gcc")
    env = dict(os.environ, PIC_ORACLE_SANITIZE="1", LD_PRELOAD=asan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    cmd = [sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider",
           os.path.join(ROOT, "tests", "test_oracle_pins.py"),
           os.path.join(ROOT, "tests", "test_sensitivity.py")]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    tail = (r.stdout + r.stderr)[-4000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "failed" not in r.stdout, tail
    assert "ERROR: AddressSanitizer" not in tail and "runtime error:" not in tail, tail
    # the sanitized build is the one that ran
    assert os.path.exists(os.path.join(ROOT, "oracle", "libpic_oracle_san.so"))
