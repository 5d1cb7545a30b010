"""Builds libwtide.so in-tree with nvcc for sm_100a (no torch, no JIT cache).

    python -m paper_2605_13987_b200.build
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["csrc/geometry.cpp", "csrc/solve.cu", "csrc/conv.cu"]
DEPS = SOURCES + ["csrc/fft.cuh", "csrc/regfft.cuh", "csrc/solve_common.cuh", "csrc/solve_boundary.cuh",
                  "csrc/solve_generic.cuh", "csrc/solve_fast.cuh", "csrc/geometry.h", "../include/wtide.h"]
LIB = os.path.join(HERE, "libwtide.so")


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, d)) > t for d in DEPS)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-shared", "-Xcompiler", "-fPIC", "-O3", "-std=c++17", "-lineinfo",
           "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static",
           "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
