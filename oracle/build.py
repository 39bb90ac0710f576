"""Build the CPU oracle (test infrastructure): gcc -> oracle/libsteps_oracle.so.

Usage: python oracle/build.py        (also called by __graft_entry__.build()).
Building the checker is not using it; nothing in the product path loads this library."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "steps_oracle.c")
LIB = os.path.join(HERE, "libsteps_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -O2, no -ffast-math: the compensated summation must survive.  -march is left at the
    # baseline so a library built on one box runs on the GPU box's host CPU.
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
