"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (the oracle is the
reference every parity claim rests on, so its own memory safety and arithmetic are checked once).

A child python runs the hand-computed pins, the golden fixtures and a slice of the brute-force pins against
oracle/libfestina_oracle_san.so (same source, -fsanitize=address,undefined -fno-sanitize-recover=undefined) with
libasan preloaded; any report aborts the child."""
from __future__ import annotations

import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _runtime(name: str) -> str:
    p = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else ""


def test_oracle_pins_under_asan_ubsan():
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan:
        pytest.skip("gcc's libasan.so is not installed")
    env = dict(os.environ, FESTINA_ORACLE_SANITIZE="1", LD_PRELOAD=" ".join(x for x in (asan, ubsan) if x),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", PYTHONMALLOC="malloc")
    sel = ("by_hand or bump or idle_decode or cold_start or fig6 or fig8 or appendix_g or margin or slot_rule "
           "or duplicate or inactive or (bruteforce_tiny and (0 or 2 or 5))")
    files = [os.path.join(ROOT, "tests", f) for f in
             ("test_oracle_pins.py", "test_golden.py", "test_oracle_dispatch.py", "test_oracle_commit.py",
              "test_oracle_batching.py", "test_oracle_alg1.py", "test_oracle_plan.py", "test_oracle_migration.py")]
    p = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-k",
                        f"({sel}) or golden or dispatch or commit or batching or alg1 or plan or migration"] + files,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    tail = (p.stdout + p.stderr)[-4000:]
    assert p.returncode == 0, tail
    assert "passed" in p.stdout and "ERROR: AddressSanitizer" not in tail and "runtime error" not in tail, tail
