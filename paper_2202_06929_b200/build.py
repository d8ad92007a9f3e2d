"""Compile the CUDA sources under csrc/ into libfrnn_b200.so (in-tree, sm_100a only)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfrnn_b200.so")
SOURCES = [os.path.join(CSRC, "frnn.cu"), os.path.join(CSRC, "frnn_next.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "frnn_kernels.cuh"), os.path.join(CSRC, "launch_plan.h"), os.path.join(HERE, "..", "include", "frnn.h")]
# No --use_fast_math: the d2 chain is written with explicit rounding intrinsics and denormals must
# not be flushed (R3).
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "--extended-lambda",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + f".{os.getpid()}.tmp"
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("FRNN_NVCC_EXTRA", "").split()          # e.g. -DFRNN_SEARCH_MIN_BLOCKS=4 for sweeps
    res = subprocess.run([nvcc, *NVCC_FLAGS, *extra, *SOURCES, "-o", tmp], capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
