"""SURVEY.md section 5, sanitizer row (CPU side): the oracle built with AddressSanitizer + UndefinedBehaviorSanitizer
runs its pins clean, and the host runtime's validation paths (no GPU needed) run clean under the same preload.

The sanitized oracle is a second library (oracle/liborchard_oracle_san.so, selected by ORCHARD_ORACLE_SANITIZE=1); the
pins run in a child process under LD_PRELOAD=libasan.so.  UBSan is built with -fno-sanitize-recover, ASan aborts on its
first report, so a finding is a non-zero exit code.  Leak checking is off: CPython itself never frees everything."""
from __future__ import annotations

import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _asan_runtime():
    p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    return os.path.realpath(p) if os.path.isabs(p) and os.path.exists(p) else None


def _run(args, extra_env):
    rt = _asan_runtime()
    if rt is None:
        pytest.skip("gcc has no libasan.so on this machine")
    env = dict(os.environ, LD_PRELOAD=rt, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:exitcode=97",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", **extra_env)
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-p", "no:cacheprovider"] + args,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    out = r.stdout + r.stderr
    assert "runtime error:" not in out and "AddressSanitizer" not in out, out[-4000:]
    assert r.returncode == 0, out[-4000:]
    return out


# the pins that touch every allocation pattern of the oracle: events (empty and non-empty drains), wrenches, apples,
# randomization of materials and geometry, state / counter round trips, the PCG mode, friction / drag / rails
ORACLE_PINS = ("config1_events or wrench_slot or state_round_trip or pcg_equals_cholesky or geometry_randomization or "
               "post_rupture or snapped or force_rails or resets_on_a_miss or precedence or virtual_mass or "
               "randomize_draws or ternary")


def test_oracle_pins_run_clean_under_asan_and_ubsan():
    out = _run(["tests/test_oracle_pins.py", "-k", ORACLE_PINS], {"ORCHARD_ORACLE_SANITIZE": "1", "OMP_NUM_THREADS": "2"})
    assert " passed" in out and "failed" not in out


def test_host_validation_paths_run_clean_under_asan():
    """libob.so is not instrumented (nvcc build), but ASan's allocator and interceptors still see every malloc / memcpy
    the host runtime makes on the paths that need no GPU: ob_workspace_bytes, the validation errors, the no-device
    refusal of ob_create."""
    out = _run(["tests/test_abi.py"], {})
    assert " passed" in out and "failed" not in out
