"""AddressSanitizer + UndefinedBehaviorSanitizer over the oracle (oracle/cosmo_oracle.c) and over the CUDA path's per-element headers
compiled for the host (tests/hostcheck/hostcheck.cpp), on seeded stress inputs: config 5 with its structured blocks, the extra-w mix,
two-limit pairs.  compute-sanitizer is closed on the GPU pool, so this host run, the parity tests and the
library's own argument checks are what guards memory safety of the arithmetic code."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HC = os.path.join(ROOT, "tests", "hostcheck")


def _runtime(name):
    p = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_and_host_math_under_asan_ubsan():
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("sanitizer runtimes not installed")
    flags = ["-O1", "-g", "-fPIC", "-shared", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    lo, lh = os.path.join(HC, "liboracle_asan.so"), os.path.join(HC, "libhostcheck_asan.so")
    subprocess.run(["gcc", "-std=gnu11", "-fopenmp"] + flags + ["-o", lo, os.path.join(ROOT, "oracle", "cosmo_oracle.c"), "-lm"], check=True)
    subprocess.run(["g++", "-std=c++17", "-ffp-contract=off", "-Wno-unknown-pragmas"] + flags + ["-o", lh, os.path.join(HC, "hostcheck.cpp")], check=True)
    env = dict(os.environ, LD_PRELOAD=f"{asan}:{ubsan}", ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", OMP_NUM_THREADS="4")
    r = subprocess.run([sys.executable, os.path.join(HC, "sanitized_run.py"), lo, lh], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "sanitized run finished" in r.stdout and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
