"""SURVEY.md section 5 (race detection / sanitizers): the CPU oracle and the production CPU fast marching are compiled
with AddressSanitizer + UndefinedBehaviorSanitizer into one executable with tests/sanitize/driver.cpp, which runs
their FMM / back-projection paths on small edge-case problems.  Any sanitizer report aborts the run."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]


@pytest.mark.skipif(shutil.which("gcc") is None or shutil.which("g++") is None, reason="needs gcc / g++")
def test_oracle_and_production_fmm_under_asan_ubsan(tmp_path):
    obj_oracle = str(tmp_path / "pat_oracle.o")
    obj_fmm = str(tmp_path / "fmm.o")
    exe = str(tmp_path / "sanitize_driver")
    # the oracle with ITS flags (-ffp-contract=off is part of its definition) plus the sanitizers
    subprocess.run(["gcc", "-std=c11", "-ffp-contract=off", "-fopenmp", *SAN, "-c", os.path.join(ROOT, "oracle", "pat_oracle.c"),
                    "-o", obj_oracle], check=True)
    subprocess.run(["g++", "-std=c++17", "-fopenmp", *SAN, "-c",
                    os.path.join(ROOT, "paper_1501_03869_b200", "csrc", "fmm.cpp"), "-o", obj_fmm], check=True)
    subprocess.run(["g++", "-std=c++17", "-fopenmp", *SAN, os.path.join(ROOT, "tests", "sanitize", "driver.cpp"),
                    obj_oracle, obj_fmm, "-o", exe, "-lm"], check=True)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:halt_on_error=1:abort_on_error=0",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="3")
    r = subprocess.run([exe], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, "sanitizer driver failed:\n%s\n%s" % (r.stdout[-2000:], r.stderr[-6000:])
    assert "sanitizer driver: ok" in r.stdout
