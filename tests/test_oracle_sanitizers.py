"""SURVEY.md section 5, sanitizer leg: the graded oracle (oracle/psync_oracle.cpp) built with
-fsanitize=address,undefined and its own pin tests run against that build in a subprocess (the ASan runtime has to be
the first library of the process, hence LD_PRELOAD).  Any out-of-bounds access, use-after-free, signed overflow, bad
shift or misaligned access in the oracle aborts the subprocess and fails this test.  (compute-sanitizer for the CUDA
side is closed on this GPU pool; guard-band tests in tests/test_gpu_update.py stand in for it.)"""
import os
import subprocess
import sys

import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
PIN_FILES = ["test_oracle_select.py", "test_oracle_update.py", "test_oracle_per_server.py", "test_oracle_async.py",
             "test_oracle_helpers.py", "test_oracle_stragglers.py", "test_oracle_slices.py",
             "test_oracle_staleness.py"]


def _runtime(name):
    path = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return path if os.path.isabs(path) and os.path.exists(path) else None


def test_oracle_pins_pass_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if asan is None:
        pytest.skip("no libasan.so beside gcc")
    lib = oracle.build_sanitized(tmp_path)
    env = dict(os.environ)
    env["PSYNC_ORACLE_LIB"] = str(lib)
    env["LD_PRELOAD"] = ":".join(p for p in (asan, ubsan) if p)
    env["ASAN_OPTIONS"] = "detect_leaks=0:abort_on_error=1:halt_on_error=1"     # CPython itself "leaks" by design
    env["UBSAN_OPTIONS"] = "halt_on_error=1:print_stacktrace=1"
    env["OMP_NUM_THREADS"] = "4"
    files = [os.path.join(HERE, f) for f in PIN_FILES if os.path.exists(os.path.join(HERE, f))]
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", *files],
                       env=env, capture_output=True, text=True, cwd=os.path.dirname(HERE), timeout=900)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "ERROR: AddressSanitizer" not in tail and "runtime error" not in tail, tail
    # the run really used the instrumented build
    probe = subprocess.run([sys.executable, "-c",
                            "import oracle, ctypes; L = oracle.lib(); print(L._name)"],
                           env=env, capture_output=True, text=True, cwd=os.path.dirname(HERE))
    assert "libpsync_oracle_asan.so" in probe.stdout, probe.stdout + probe.stderr
