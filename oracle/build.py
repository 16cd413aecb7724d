"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not the product).

    python oracle/build.py        -> oracle/libafid_ref.so

gcc -O2 -ffp-contract=off (no FMA contraction, no fast-math: DESIGN.md R16), OpenMP over
independent lines / systems only.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "afid_ref.c")
LIB = os.path.join(HERE, "libafid_ref.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-shared", "-fPIC", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
