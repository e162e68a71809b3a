"""Build the CPU oracle (test infrastructure) into oracle/libmpm_oracle.so with gcc.

-O2, no FMA contraction, no fast-math: the arithmetic is exactly what mpm_oracle.c spells out.
Usage: python oracle/build.py   (also called by __graft_entry__.build() and tests/conftest.py)
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mpm_oracle.c")
HDR = os.path.join(HERE, "mpm_oracle.h")
LIB = os.path.join(HERE, "libmpm_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
