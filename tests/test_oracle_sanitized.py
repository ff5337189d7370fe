"""the oracle built with -fsanitize=address,undefined and every pin of
tests/test_oracle_pins.py (P1-P10, N3) re-run on that build.  The sanitizer runtime has to be the first
library of the process, so the pins run in a subprocess with libasan preloaded; any out-of-bounds access,
use of uninitialised stack, signed overflow or misaligned access in oracle/stag_oracle.cpp aborts it."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _runtime(name):
    try:
        p = subprocess.check_output(["g++", "-print-file-name=" + name], text=True).strip()
    except Exception:
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_pins_under_asan_ubsan():
    asan = _runtime("libasan.so")
    if asan is None:
        pytest.skip("g++ has no libasan here")
    env = dict(os.environ)
    env.update(STAG_ORACLE_SANITIZE="1", LD_PRELOAD=asan,
               ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                        os.path.join(ROOT, "tests", "test_oracle_pins.py")],
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "ERROR: AddressSanitizer" not in tail and "runtime error" not in tail, tail
    # the sanitized library really was the one loaded
    assert os.path.exists(os.path.join(ROOT, "oracle", "libstag_oracle_san.so"))
