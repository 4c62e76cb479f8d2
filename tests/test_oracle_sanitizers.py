"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer: a small case through every oracle
entry point -- brute force, cell list, time stepping with walls, reflection, thermostat and prism pore -- must run clean."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_sanitize")
    cmd = ["gcc", "-O1", "-g", "-ffp-contract=off", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fopenmp",
           "-std=c11", os.path.join(HERE, "oracle_sanitize_main.c"), "-o", exe, "-lm"]
    built = subprocess.run(cmd, capture_output=True, text=True)
    if built.returncode != 0 and "asan" in (built.stderr or "").lower():
        pytest.skip("libasan is not installed: " + built.stderr.splitlines()[-1])
    assert built.returncode == 0, built.stderr
    env = dict(os.environ, OMP_NUM_THREADS="2", ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    run = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=120)
    assert run.returncode == 0, run.stdout + run.stderr
    assert run.stdout.startswith("ok ") and "runtime error" not in run.stderr and "AddressSanitizer" not in run.stderr
