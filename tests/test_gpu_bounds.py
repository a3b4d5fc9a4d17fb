"""Memory-safety check of the CUDA path without compute-sanitizer (not available on the build pool):
the same sources compiled with -DGALE_CHECK_BOUNDS=1 (libgale_checked.so) verify every tile against the
launch's shared-memory capacities and every computed staging index before it is written, and report
through the device error word. The negative control understates one capacity and must be detected."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(extra_env):
    from paper_2507_15230_b200.build import build_library
    lib = build_library(checked=True)
    env = dict(os.environ, GALE_LIBRARY=lib, **extra_env)
    return subprocess.run([sys.executable, os.path.join(ROOT, "tests", "bounds_runner.py")], env=env,
                          capture_output=True, text=True, timeout=900)


def test_bounds_checked_build_is_clean_and_bit_exact():
    r = _run({})
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "ALL CHECKED CASES PASSED" in r.stdout and r.stdout.count("\nok ") + r.stdout.startswith("ok ") >= 24


def test_bounds_checker_fires_on_understated_capacity():
    r = _run({"GALE_CHECK_SELFTEST": "1"})
    assert r.returncode not in (0, 3), r.stdout[-1000:]            # 3 = ran through without detection
    assert "GALE_ERR_WORKSPACE" in r.stderr and "guard fired" in r.stderr, r.stderr[-1500:]
