"""Build paper_2606_11867_b200/libforemoe.so (the C-ABI library of include/foremoe.h) with nvcc for
sm_100a.  In-tree on purpose: the built .so travels to the GPU box with the repo snapshot.

    python -m paper_2606_11867_b200.build [--force] [-v] [--tuning]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libforemoe.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
         "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [
        os.path.join(HERE, "..", "include", "foremoe.h"), os.path.abspath(__file__)]
    return any(os.path.getmtime(p) > t for p in deps)


LIB_TUNING = os.path.join(HERE, "libforemoe_tuning.so")


def build(force: bool = False, verbose: bool = False, tuning: bool = False) -> str:
    """Compile every .cu under csrc/ into libforemoe.so; returns its path.

    tuning=True builds libforemoe_tuning.so instead, with -DFOREMOE_TUNING: the same kernels with
    mutable launch parameters and the extra export foremoe_tuning_set (sweeps only; the binding
    never loads it)."""
    if tuning:
        return _build(LIB_TUNING, "build_tuning", ["-DFOREMOE_TUNING"], verbose)
    if not force and not _stale():
        return LIB
    return _build(LIB, "build", [], verbose)


def _build(LIB: str, objdir: str, extra, verbose: bool) -> str:
    objs = []
    procs = []
    os.makedirs(os.path.join(HERE, objdir), exist_ok=True)
    for src in sources():
        obj = os.path.join(HERE, objdir, os.path.basename(src)[:-3] + ".o")
        cmd = [NVCC] + [f for f in FLAGS if f != "-shared"] + list(extra) + ["-c", src, "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(obj)
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    link = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
            "-o", LIB + ".tmp"] + objs
    subprocess.run(link, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, tuning="--tuning" in sys.argv))
