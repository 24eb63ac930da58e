"""The FP64 oracle (oracle/pdm_oracle.c) built with -fsanitize=address,undefined and run on ragged
cases by a small C driver (tests/oracle_sanitize_main.c).  CPU only ("oracle
built with -fsanitize=address,undefined").  Catches out-of-bounds reads at the zero edges (R5),
index overflow before the clamp, and misuse of the per-thread accumulators."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


@pytest.mark.skipif(shutil.which("gcc") is None, reason="gcc not available")
def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    exe = tmp_path / "oracle_sanitize"
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-fopenmp", "-ffp-contract=off",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer",
           os.path.join(ROOT, "oracle", "pdm_oracle.c"), os.path.join(HERE, "oracle_sanitize_main.c"),
           "-o", str(exe), "-lm"]
    build = subprocess.run(cmd, capture_output=True, text=True)
    if build.returncode != 0 and ("asan" in build.stderr.lower() or "ubsan" in build.stderr.lower()):
        pytest.skip("sanitizer runtime libraries are not installed: " + build.stderr[-200:])
    assert build.returncode == 0, build.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", OMP_NUM_THREADS="3",
               UBSAN_OPTIONS="print_stacktrace=1")
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=120)
    assert run.returncode == 0, (run.stdout, run.stderr)
    assert "AddressSanitizer" not in run.stderr and "runtime error" not in run.stderr, run.stderr
    assert run.stdout.count("rc=0") == 5, run.stdout
