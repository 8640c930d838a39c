"""Build oracle/libjenga_oracle.so (test infrastructure; see jenga_oracle.c header).

    python oracle/build.py

-ffp-contract=off: no fused multiply-add, so every fp64 operation rounds separately;
the CUDA broadphase's fp64 re-check relies on this to reproduce Eq. 10 decisions exactly.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "jenga_oracle.c")
LIB = os.path.join(HERE, "libjenga_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wno-misleading-indentation", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
