"""The C ABI driven from plain C (tests/c_abi_smoke.c): no Python, torch or CUDA headers on the caller's side.
CPU: the program compiles and links against liblgf.so with nothing but include/lgf.h.  GPU: it runs and its
closed-form checks (constant fields: theta = 0, F = (1/12) sum Re Tr V_mu, fixed point of the iteration) pass."""
import os
import subprocess

import pytest

import paper_1208_1186_b200 as lgf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _build(tmp_path):
    libdir = os.path.dirname(lgf.library_path())
    exe = str(tmp_path / "c_abi_smoke")
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-Wextra", "-Werror", "-I", os.path.join(ROOT, "include"),
           os.path.join(ROOT, "tests", "c_abi_smoke.c"), "-o", exe, "-L", libdir, "-llgf", "-lm",
           "-Wl,-rpath," + libdir, "-Wl,-rpath,/usr/local/cuda/lib64"]
    subprocess.run(cmd, check=True)
    return exe


def test_c_program_compiles_against_the_header(tmp_path):
    lgf.load_library()          # raises if liblgf.so is missing
    assert os.path.exists(_build(tmp_path))


@pytest.mark.gpu
def test_c_program_runs(tmp_path):
    exe = _build(tmp_path)
    p = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stdout + p.stderr
    assert "c_abi_smoke: ok" in p.stdout
