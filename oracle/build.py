"""Compile oracle/foremoe_oracle.c into oracle/liboracle_foremoe.so with gcc.

TEST INFRASTRUCTURE: building the checker is not using it.  -ffp-contract=off keeps the
compiler from fusing or re-associating any floating point (the only fused op is the explicit
fmaf of O6); no -ffast-math, no intrinsics, no OpenMP.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "foremoe_oracle.c")
LIB = os.path.join(HERE, "liboracle_foremoe.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-ffp-contract=off", "-Wall",
           "-Wextra", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
