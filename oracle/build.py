"""Build the CPU oracle (test infrastructure): gcc -> oracle/libsteps_oracle.so.

Usage: python oracle/build.py        (also called by __graft_entry__.build()).
Building the checker is not using it; nothing in the product path loads this library.

Flags: -O3 -march=native -fopenmp, as BASELINE.md's CPU-baseline plan states, with -ffp-contract=off and no
-ffast-math so that the arithmetic (and the compensated summation) is the source's, operation by operation.
-march=native ties the binary to the host CPU, and the built library travels between boxes with the working tree,
so the CPU's feature flags are recorded beside it and the library is rebuilt when they differ."""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "steps_oracle.c")
LIB = os.path.join(HERE, "libsteps_oracle.so")
STAMP = LIB + ".host"
CFLAGS = ["-O3", "-march=native", "-ffp-contract=off", "-std=c11", "-fopenmp", "-fPIC", "-shared"]


def host_tag() -> str:
    """Hash of this host's CPU feature flags (what -march=native resolves to)."""
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith(("flags", "Features")):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha256((flags + " ".join(CFLAGS)).encode()).hexdigest()[:16]


def build(force: bool = False) -> str:
    tag = host_tag()
    fresh = os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)
    try:
        same_host = open(STAMP).read().strip() == tag
    except OSError:
        same_host = False
    if not force and fresh and same_host:
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"])
    os.replace(tmp, LIB)
    with open(STAMP, "w") as f:
        f.write(tag + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
