"""The boundary used from plain C (no Python, no torch in the caller): tests/c_abi_demo.c is compiled
with gcc against include/foremoe.h, linked with libforemoe.so and the CUDA runtime, and run."""
import os
import subprocess

import pytest

from paper_2606_11867_b200 import build as fbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _compile(tmp_path):
    lib = fbuild.build()
    exe = tmp_path / "c_abi_demo"
    subprocess.run(["gcc", "-std=c11", "-O1", "-Wall", "-Wextra", "-Werror",
                    "-I", os.path.join(ROOT, "include"), "-I", os.path.join(CUDA, "include"),
                    os.path.join(ROOT, "tests", "c_abi_demo.c"), "-o", str(exe),
                    lib, "-L", os.path.join(CUDA, "lib64"), "-lcudart",
                    "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.join(CUDA, "lib64")], check=True)
    return exe


def test_c_caller_compiles_and_links(tmp_path):
    """No GPU needed: the C caller builds against the header and links against the library."""
    assert os.path.exists(_compile(tmp_path))


@pytest.mark.gpu
def test_c_caller_runs(cuda_device, tmp_path):
    out = subprocess.run([str(_compile(tmp_path))], capture_output=True, text=True)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "c_abi_demo ok" in out.stdout
