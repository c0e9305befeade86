"""the oracle under AddressSanitizer + UndefinedBehaviorSanitizer (no GPU).

oracle/sanitize_check.c calls every function of oracle/rmsynth_oracle.c on exactly-sized heap buffers with edge
shapes; here it is compiled with the sanitizers and run.  Memory safety and undefined behaviour only -- the values are
the business of tests/test_oracle_pins.py."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    gcc = shutil.which("gcc")
    if not gcc:
        pytest.skip("gcc not available")
    exe = str(tmp_path / "sanitize_check")
    cmd = [gcc, "-O1", "-g", "-std=c11", "-fopenmp", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-fno-omit-frame-pointer", os.path.join(ROOT, "oracle", "sanitize_check.c"),
           os.path.join(ROOT, "oracle", "rmsynth_oracle.c"), "-lm", "-o", exe]
    build = subprocess.run(cmd, capture_output=True, text=True)
    if build.returncode != 0 and "sanitize" in (build.stderr or "").lower() and "cannot find" in build.stderr.lower():
        pytest.skip("sanitizer runtime libraries not installed: " + build.stderr[-200:])
    assert build.returncode == 0, build.stderr[-2000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="2")
    run = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=120)
    assert run.returncode == 0 and "sanitize_check ok" in run.stdout, (run.stdout + run.stderr)[-3000:]
