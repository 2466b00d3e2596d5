"""The boundary is a C ABI: include/bltc.h must compile as plain C and the library must be usable without Python
or torch.  tests/c_abi_smoke.c is compiled with gcc against libbltc.so and run (host-only here, full path on GPU)."""
import os
import shutil
import subprocess

import pytest

from paper_2003_01833_b200 import build as _build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _compile(tmp_path):
    lib = _build.build()
    exe = str(tmp_path / "c_abi_smoke")
    libdir = os.path.dirname(lib)
    cmd = ["gcc", "-std=c11", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
           os.path.join(ROOT, "tests", "c_abi_smoke.c"), "-o", exe, "-L", libdir, "-lbltc", "-lm",
           "-Wl,-rpath," + libdir]
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    assert r.returncode == 0, r.stdout
    return exe


@pytest.mark.skipif(shutil.which("gcc") is None, reason="gcc not on PATH")
def test_header_compiles_as_c_and_host_calls_work(tmp_path):
    exe = _compile(tmp_path)
    r = subprocess.run([exe], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=120)
    assert r.returncode == 0 and "c_abi_smoke ok" in r.stdout, r.stdout


@pytest.mark.gpu
def test_c_program_runs_the_hot_path_on_the_gpu(tmp_path):
    exe = _compile(tmp_path)
    r = subprocess.run([exe, "gpu"], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, timeout=300)
    assert r.returncode == 0 and "c_abi_smoke ok" in r.stdout, r.stdout
