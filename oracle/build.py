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


LIB32 = os.path.join(HERE, "libjenga_oracle32.so")


def build(force: bool = False, bits: int = 64) -> str:
    """bits = 32: the fp32 build of the same source (control experiment of oracle/oracle32.py only)."""
    lib = LIB if bits == 64 else LIB32
    if (not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wno-misleading-indentation", "-o", lib, SRC, "-lm"]
    if bits == 32:
        cmd[1:1] = ["-DORC_REAL_FLOAT", "-fsingle-precision-constant", "-Wno-overflow"]
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
    print(build(force="--force" in sys.argv, bits=32))
