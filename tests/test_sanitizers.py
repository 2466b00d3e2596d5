"""SURVEY.md 5 (race / memory-error detection): the host plan builder of the product (plan_host.cpp) and the CPU oracle
(oracle/*.c) built with AddressSanitizer + UndefinedBehaviorSanitizer and run on small clouds that take the odd paths.
compute-sanitizer is closed on this GPU pool (profiles/), so this is the memory-error check that can run."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(shutil.which("g++") is None, reason="g++ not on PATH")
def test_plan_builder_and_oracle_are_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "sanitize_driver")
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g", "-O1"]
    objs = []
    for src in ("direct_sum.c", "coulomb_sum.c", "bltc_cpu.c"):
        o = str(tmp_path / (src + ".o"))
        r = subprocess.run(["gcc", "-std=c11", *san, "-fopenmp", "-ffp-contract=off", "-c",
                            os.path.join(ROOT, "oracle", src), "-o", o], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        assert r.returncode == 0, r.stdout
        objs.append(o)
    r = subprocess.run(["g++", "-std=c++17", *san, "-fopenmp", "-pthread", "-ffp-contract=off",
                        os.path.join(ROOT, "tests", "sanitize_driver.cpp"),
                        os.path.join(ROOT, "paper_2003_01833_b200", "csrc", "plan_host.cpp"), *objs, "-o", exe, "-lm"],
                       stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert r.returncode == 0, r.stdout
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([exe], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=600)
    assert r.returncode == 0 and "sanitize ok" in r.stdout, r.stdout[-4000:]
    assert "runtime error" not in r.stdout and "AddressSanitizer" not in r.stdout, r.stdout[-4000:]
