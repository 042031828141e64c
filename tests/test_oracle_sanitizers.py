"""CPU: the oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY section 5 "race detection /
sanitizers": "ASan/UBSan on the oracle").  tests/host/oracle_sanitize.c drives every oracle entry point on small
ragged problems; the build aborts on the first finding (-fno-sanitize-recover=all), leaks included."""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _build(tmp_path, extra):
    exe = str(tmp_path / "oracle_sanitize")
    cmd = ["gcc", "-std=c11", "-O1", "-g", "-fno-omit-frame-pointer", "-ffp-contract=off", "-mfma",
           "-Wall", "-Wextra", "-Wno-unknown-pragmas"] + extra + [
        "-o", exe, os.path.join(ROOT, "tests", "host", "oracle_sanitize.c"),
        os.path.join(ROOT, "oracle", "sldg_oracle.c"), "-lm"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and "sanitize" in r.stderr and "cannot find" in r.stderr:
        pytest.skip("sanitizer runtime not installed: " + r.stderr.strip().splitlines()[-1])
    assert r.returncode == 0, r.stderr
    return exe


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    exe = _build(tmp_path, ["-fsanitize=address,undefined", "-fno-sanitize-recover=all"])
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert "oracle sanitizer run: ok" in r.stdout


def test_oracle_openmp_build_is_clean_under_ubsan(tmp_path):
    """The build the tests actually use (OpenMP over lines) under UBSan, 4 threads."""
    exe = _build(tmp_path, ["-fopenmp", "-fsanitize=undefined", "-fno-sanitize-recover=all"])
    env = dict(os.environ, OMP_NUM_THREADS="4")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
