"""Compile oracle/frnn_oracle.c into oracle/libfrnn_oracle.so with gcc (no CUDA, no torch).

TEST INFRASTRUCTURE ONLY -- see the header of frnn_oracle.c.  Flags follow DESIGN.md section 3:
-ffp-contract=off so the only fused multiply-add is the explicit fmaf(); never -ffast-math.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "frnn_oracle.c")
LIB = os.path.join(HERE, "libfrnn_oracle.so")
FLAGS = ["-O2", "-std=c11", "-fopenmp", "-mfma", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-Wall"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".{os.getpid()}.tmp"
    subprocess.run(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
