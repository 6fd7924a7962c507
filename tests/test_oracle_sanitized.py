"""SURVEY section 5 / VERDICT r1 item 8: the host oracle under AddressSanitizer + UndefinedBehaviorSanitizer.

compute-sanitizer is closed on the GPU pool, but the oracle is plain C and needs no GPU: this test rebuilds
oracle/game_oracle.c with -fsanitize=address,undefined (GAME_ORACLE_SANITIZE=1 selects that build in oracle/oracle.py)
and re-runs the oracle pin suite (P1-P24, the tied families and the exact pins) against it in a child pytest with the
sanitizer runtimes preloaded.  Any out-of-bounds access, use-after-free, signed overflow, misaligned access or invalid
shift in the oracle aborts the child with a non-zero exit code.
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PIN_FILES = ["tests/test_oracle_expansion.py", "tests/test_oracle_fitness.py", "tests/test_oracle_rng_ga.py",
             "tests/test_oracle_tied.py", "tests/test_oracle_exact_pins.py"]


def _runtime(name):
    out = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


def test_oracle_pins_under_asan_ubsan():
    if os.environ.get("GAME_ORACLE_SANITIZE") == "1":
        pytest.skip("already inside the sanitized child run")
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc sanitizer runtimes not installed")
    env = dict(os.environ)
    env.update(GAME_ORACLE_SANITIZE="1", LD_PRELOAD=asan + ":" + ubsan,
               # CPython's allocator and torch's static initialisers are not what is being checked: no leak report
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4")
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider"] + PIN_FILES, cwd=ROOT, env=env,
                       capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, "sanitized oracle run failed:\n" + tail
    assert "passed" in r.stdout and "AddressSanitizer" not in tail and "runtime error" not in tail, tail
    # the child really loaded the instrumented library
    assert os.path.exists(os.path.join(ROOT, "oracle", "libgame_oracle_san.so"))
