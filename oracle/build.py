"""Build the C oracle (TEST INFRASTRUCTURE ONLY) into oracle/libte_oracle.so with gcc.

Flags follow DESIGN.md reading 16: -O2 -fno-fast-math -ffp-contract=off (no FMA contraction, so the
oracle's rounding does not depend on the compiler's fusion choices), OpenMP for the pair / bra loops.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "te_oracle.c")
LIB = os.path.join(HERE, "libte_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wno-unused-function", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
