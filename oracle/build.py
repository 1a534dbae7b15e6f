"""Build the CPU oracle shared libraries (test infrastructure, see md_oracle.c header).

    python -m oracle.build          # libmd_oracle.so (double) and libmd_oracle_quad.so (__float128)
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "md_oracle.c")
LIB = os.path.join(HERE, "libmd_oracle.so")
LIB_QUAD = os.path.join(HERE, "libmd_oracle_quad.so")


def _stale(target):
    return not os.path.exists(target) or os.path.getmtime(target) < os.path.getmtime(SRC)


def build(force=False, quad=True):
    """gcc -O2, no fast-math, OpenMP over quartets (CPU-baseline plan)."""
    base = ["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-Wall", SRC]
    if force or _stale(LIB):
        subprocess.check_call(base + ["-o", LIB, "-lm"])
    if quad and (force or _stale(LIB_QUAD)):
        subprocess.check_call(base + ["-DORACLE_QUAD", "-o", LIB_QUAD, "-lquadmath", "-lm"])
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print(LIB)
