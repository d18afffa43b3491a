"""Build the CPU oracle (test infrastructure) into oracle/libocfd_oracle.so.

    python oracle/build.py

Flags follow DESIGN.md section 4: -O2, no FMA contraction, no fast-math, OpenMP over outer loops.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ocfd_oracle.c")
LIB = os.path.join(HERE, "libocfd_oracle.so")


def build(force=False):
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-std=c11", SRC, "-o", LIB, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
