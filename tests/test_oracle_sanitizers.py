"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: the pins of every oracle function
are re-run in a child process against liboracle_san.so (gcc -fsanitize=address,undefined); any out-of-bounds access,
use after free, signed overflow, misaligned or invalid load in oracle/vg_oracle.c aborts that process."""
import os
import subprocess
import sys

import pytest

from oracle import build as oracle_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PINS = ["tests/test_oracle_pins.py", "tests/test_oracle_nav.py", "tests/test_oracle_boolean.py", "tests/test_oracle_world.py",
        "tests/test_oracle_surface.py"]


def test_oracle_pins_pass_under_asan_and_ubsan():
    rt = oracle_build.asan_runtime()
    if not os.path.isabs(rt) or not os.path.exists(rt):
        pytest.skip("no libasan.so next to this gcc")
    oracle_build.build_sanitized()
    env = dict(os.environ, ORACLE_SANITIZE="1", LD_PRELOAD=rt, ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4")
    # the marching / sampling pins call the same C entry points as the others, thousands of times from numpy loops: they
    # run under the sanitizers only with VG_SANITIZE_FULL=1 (6 minutes; done once per round)
    quick = [] if os.environ.get("VG_SANITIZE_FULL") == "1" else ["-k", "not marching and not brute_force and not sphere_tracing and not sampling"]
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"] + quick + PINS,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "runtime error" not in r.stdout + r.stderr and "AddressSanitizer" not in r.stdout + r.stderr, tail
    assert " passed" in r.stdout
