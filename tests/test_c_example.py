"""The boundary is a C ABI: include/swe_b200.h compiles as strict C99 and examples/dam_break.c (plain
C, no Python, no torch) links against libswe_b200.so.  Without a GPU the program fails loudly at
swe_mesh_create; on the GPU box it runs the dam break and checks mass conservation itself."""
import os
import subprocess

import pytest

import paper_2307_16758_b200 as sw

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_2307_16758_b200")


def _build(tmp_path):
    sw.lib()                                            # makes sure the library is built
    exe = str(tmp_path / "dam_break")
    cmd = ["gcc", "-std=c99", "-O2", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
           os.path.join(ROOT, "examples", "dam_break.c"), "-L", PKG, "-lswe_b200", "-Wl,-rpath," + PKG, "-lm", "-o", exe]
    out = subprocess.run(cmd, capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    return exe


def test_c_example_compiles_links_and_fails_loudly_without_a_gpu(tmp_path):
    import torch
    exe = _build(tmp_path)
    if torch.cuda.is_available():
        pytest.skip("a GPU is present: see the gpu test")
    out = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert out.returncode == 1 and "no CUDA device" in out.stderr


@pytest.mark.gpu
def test_c_example_runs_on_the_gpu(tmp_path):
    exe = _build(tmp_path)
    out = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "HLLC" in out.stdout and "MUSCL-RK2" in out.stdout and "mass drift" in out.stdout
    assert "8 zones x 2 layers" in out.stdout and "bit-identical to the un-zoned run" in out.stdout
