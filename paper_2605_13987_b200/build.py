"""Builds libwtide.so in-tree with nvcc for sm_100a (no torch, no JIT cache).

    python -m paper_2605_13987_b200.build [--force] [-v]

Each translation unit is compiled to an object under build/ (git-ignored) when it or one of its
headers changed, the units in parallel; the objects are then linked into libwtide.so beside this file.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
HEADERS = ["csrc/fft.cuh", "csrc/regfft.cuh", "csrc/solve_common.cuh", "csrc/solve_boundary.cuh", "csrc/solve_generic.cuh",
           "csrc/solve_fast.cuh", "csrc/solve_persistent.cuh", "csrc/solve_plan.h", "csrc/geometry.h", "../include/wtide.h"]
# translation unit -> headers it includes
UNITS = {
    "csrc/geometry.cpp": ["csrc/geometry.h", "../include/wtide.h"],
    "csrc/solve.cu": HEADERS,
    "csrc/solve_chain.cu": HEADERS,
    "csrc/solve_persistent.cu": HEADERS,
    "csrc/conv.cu": ["csrc/geometry.h", "csrc/locate.cuh", "../include/wtide.h"],
    "csrc/next.cu": ["csrc/geometry.h", "csrc/locate.cuh", "../include/wtide.h"],
    "csrc/static_field.cu": HEADERS,
    "csrc/peaks.cu": ["csrc/geometry.h", "../include/wtide.h"],
}
SOURCES = [u for u in UNITS if os.path.exists(os.path.join(HERE, u))]
DEPS = SOURCES + [h for h in HEADERS if os.path.exists(os.path.join(HERE, h))]
LIB = os.path.join(HERE, "libwtide.so")
OBJDIR = os.path.join(HERE, "build")
FLAGS = ["-Xcompiler", "-fPIC", "-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a"]


def _mtime(rel):
    p = os.path.join(HERE, rel)
    return os.path.getmtime(p) if os.path.exists(p) else 0.0


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(_mtime(d) > t for d in DEPS)


def _obj(unit):
    return os.path.join(OBJDIR, os.path.basename(unit) + ".o")


def _stale(unit):
    o = _obj(unit)
    if not os.path.exists(o):
        return True
    t = os.path.getmtime(o)
    return _mtime(unit) > t or any(_mtime(h) > t for h in UNITS[unit]) or os.path.getmtime(__file__) > t


def build(force=False, verbose=False, defines=()):
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJDIR, exist_ok=True)
    extra = (["-Xptxas=-v"] if verbose else []) + [f"-D{d}" for d in defines]

    def compile_unit(unit):
        cmd = [nvcc, "-c"] + FLAGS + extra + ["-o", _obj(unit), os.path.join(HERE, unit)]
        r = subprocess.run(cmd, cwd=HERE, capture_output=True, text=True)
        return unit, r

    todo = [u for u in SOURCES if force or defines or _stale(u)]
    with ThreadPoolExecutor(max_workers=max(1, len(todo))) as ex:
        results = list(ex.map(compile_unit, todo))
    for unit, r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {unit}:\n{r.stderr[-4000:]}")
    cmd = [nvcc, "-shared", "-Xcompiler", "-fPIC", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
           "-o", LIB] + [_obj(u) for u in SOURCES] + ["-lpthread"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    # --debug: -DWTIDE_DEBUG (clock stamps and kernel-skipping switches for timing experiments; never shipped)
    print(build(force="--force" in sys.argv or "--debug" in sys.argv, verbose="-v" in sys.argv,
                defines=("WTIDE_DEBUG",) if "--debug" in sys.argv else ()))
