"""The C++ oracle under -fsanitize=address,undefined ("oracle under -fsanitize=address,undefined"): the hand
traces A-H, the hash vectors and one brute-force differential per pin scope are replayed in a child process that loads the
instrumented build of arc_oracle.cpp (libasan preloaded).  Any out-of-bounds access, use after free, signed overflow or
misaligned access in the oracle aborts the child."""
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def test_oracle_traces_and_a_differential_under_asan_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not asan or not Path(asan).exists():
        pytest.skip("libasan.so not found")
    env = dict(os.environ, ARC_ORACLE_SANITIZE="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    sel = ("test_trace or test_paper_b2 or test_differential_cpp_vs_bruteforce_keys or hand_trace or test_held_pins_differential "
           "or test_step_wide_pins_differential or test_errors_leave or test_empty_and_short")
    out = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "tests/test_oracle_traces.py",
                          "tests/test_oracle_semantics.py", "tests/test_oracle_hash.py", "-k", sel + " or hash or vector or closed or inject"],
                         capture_output=True, text=True, cwd=str(ROOT), env=env, timeout=900)
    tail = (out.stdout + out.stderr)[-3000:]
    assert out.returncode == 0, tail
    assert "passed" in out.stdout and "AddressSanitizer" not in tail and "runtime error" not in tail, tail
