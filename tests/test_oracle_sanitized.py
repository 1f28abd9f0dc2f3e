"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: the whole
translation unit is compiled into a small harness (tests/oracle_sanitize_main.cpp) that calls every
exported function once on an asymmetric lattice; any out-of-bounds access, use of uninitialised
stack via UB, signed overflow or misaligned access aborts it.  CPU only."""
import os
import shutil
import subprocess
import tempfile

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.mark.skipif(shutil.which("g++") is None, reason="g++ not available")
def test_oracle_runs_clean_under_asan_ubsan():
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, "oracle_sanitize")
        cmd = ["g++", "-std=c++17", "-O1", "-g", "-fopenmp", "-fsanitize=address,undefined",
               "-fno-sanitize-recover=all", "-fno-omit-frame-pointer",
               os.path.join(HERE, "oracle_sanitize_main.cpp"), "-o", exe]
        build = subprocess.run(cmd, capture_output=True, text=True)
        if build.returncode != 0 and "sanitize" in build.stderr and "cannot find" in build.stderr:
            pytest.skip("sanitizer runtime not installed")
        assert build.returncode == 0, build.stderr[-2000:]
        env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", OMP_NUM_THREADS="2")
        run = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
        assert run.returncode == 0, (run.stdout + run.stderr)[-3000:]
        assert run.stdout.count(" ok ") == 2
