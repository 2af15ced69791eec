"""ASan + UBSan pass over the oracle: oracle/foremoe_oracle.c is rebuilt with
-fsanitize=address,undefined -fno-sanitize-recover and its pins (quota, path, placement, swap, local,
backward) are run on that build in a child process (the sanitizer runtime has to be preloaded into
the interpreter).  Any out-of-bounds access, signed overflow, misaligned or invalid shift in the
checker aborts the child and fails this test."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

PINS = ["tests/test_oracle_quota.py", "tests/test_oracle_path.py", "tests/test_oracle_placement.py",
        "tests/test_oracle_swap.py", "tests/test_oracle_local.py", "tests/test_oracle_backward.py",
        "tests/test_oracle_tradeoff.py", "tests/test_oracle_replica_search.py"]


def _runtime(name):
    p = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_pins_under_asan_ubsan():
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc sanitizer runtimes not installed")
    from oracle import build as obuild
    lib = obuild.build_sanitized()
    env = dict(os.environ)
    env.update(FOREMOE_ORACLE_LIB=lib, LD_PRELOAD=asan + ":" + ubsan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", PYTHONMALLOC="malloc")
    env.pop("PYTEST_CURRENT_TEST", None)
    pins = [p for p in PINS if os.path.exists(os.path.join(ROOT, p))]
    # a quick proof that the sanitized build is the one being exercised and that it does abort
    probe = ("import ctypes, os, numpy as np; from oracle import foremoe_oracle as o; "
             "assert o.lib()._name == os.environ['FOREMOE_ORACLE_LIB']; "
             "inv = np.array([[5]], np.int32); w = np.ones((1, 1), np.float32); eo = np.zeros((1, 4), np.float32); "
             "o.combine(inv, w, eo, 1)")           # row 5 of a 1-row array: heap overflow -> ASan aborts
    r = subprocess.run([sys.executable, "-c", probe], cwd=ROOT, env=env, capture_output=True, text=True)
    assert r.returncode != 0 and "AddressSanitizer" in r.stderr, (r.returncode, r.stderr[-1500:])
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                        "-k", "not lp and not highs"] + pins,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, (r.stdout[-3000:], r.stderr[-3000:])
    assert "passed" in r.stdout
