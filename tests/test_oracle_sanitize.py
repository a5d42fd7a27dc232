"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md §5 aux row "race / memory checking"): every
scheme x lattice x boundary family with masks, porosity, the sphere with its dipole ensemble, body integrals and population
I/O, driven by tests/csrc/oracle_sanitize_main.c.  One build, one run, ~10 s."""
import os
import subprocess
import sys

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


def test_oracle_clean_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_sanitize")
    cmd = ["gcc", "-O1", "-g", "-fno-omit-frame-pointer", "-ffp-contract=off", "-fopenmp", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=all", "-Wall", os.path.join(HERE, "csrc", "oracle_sanitize_main.c"),
           os.path.join(ROOT, "oracle", "vlbm_oracle.c"), "-o", exe, "-lm"]
    b = subprocess.run(cmd, capture_output=True, text=True)
    if b.returncode != 0 and "sanitize" in b.stderr and "cannot find" in b.stderr:
        pytest.skip("libasan / libubsan not installed: " + b.stderr.splitlines()[-1])
    assert b.returncode == 0, b.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="2")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    sys.stdout.write(r.stdout)
    assert r.returncode == 0, r.stderr[-4000:]
    assert r.stdout.startswith("ok ")
    assert "ERROR" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-4000:]
