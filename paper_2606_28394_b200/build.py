"""Build csrc/libjenga.so (the C-ABI library of include/jenga.h) for sm_100a, in-tree.

    python -m paper_2606_28394_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The library is plain CUDA runtime code: no torch headers.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libjenga.so")
SOURCES = ["jenga.cu", "peaks.cu"]
DEPS = ["jenga.cu", "peaks.cu", "ksolve.cuh", "kcollide.cuh", "layout.cuh", "collide.cuh", "analysis.cuh", os.path.join("..", "..", "include", "jenga.h")]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    newest = max(os.path.getmtime(os.path.join(CSRC, d)) for d in DEPS)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = [_nvcc(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
