"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not the product).

    python -m oracle.build          # writes oracle/liboracle.so

Flags: -O2, no fast-math, -ffp-contract=off (no FMA contraction, so the R13e predicate and every
other expression is evaluated exactly as written), OpenMP over elements/states only.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dgrhd_oracle.c")
HDR = os.path.join(HERE, "dgrhd_oracle.h")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
           "-shared", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
