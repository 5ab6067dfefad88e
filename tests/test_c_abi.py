"""The C ABI from a plain C program (tests/c/abi_smoke.c): the header compiles as C and the library links (CPU check);
on a GPU box the program runs create -> wkernel_build -> grid -> dirty_image -> destroy with caller-owned workspaces
and checks counters, flux conservation and error codes itself."""
import os
import subprocess

import pytest

from paper_1905_03213_b200 import build as wbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_1905_03213_b200")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def compile_smoke(tmp_path):
    wbuild.build()
    exe = str(tmp_path / "abi_smoke")
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", "-O1", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(CUDA, "include"),
           os.path.join(ROOT, "tests", "c", "abi_smoke.c"), "-o", exe, "-L", PKG, "-lwpgrid",
           "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
           "-Wl,-rpath," + PKG, "-Wl,-rpath," + os.path.join(CUDA, "lib64")]
    subprocess.check_call(cmd)
    return exe


def test_header_compiles_as_c_and_library_links(tmp_path):
    exe = compile_smoke(tmp_path)
    assert os.path.exists(exe)


@pytest.mark.gpu
def test_c_client_runs_the_whole_path(tmp_path):
    exe = compile_smoke(tmp_path)
    out = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "abi_smoke OK" in out.stdout
