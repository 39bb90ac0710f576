"""Build the C-ABI library in-tree: nvcc (sm_100a only) -> paper_1811_05903_b200/libsteps_b200.so.

Usage: python -m paper_1811_05903_b200.build [--force] [--verbose]
nvcc cross-compiles without a GPU; the built .so travels to the GPU box with the snapshot."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsteps_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--shared", "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def deps() -> list[str]:
    return sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [
        os.path.join(os.path.dirname(HERE), "include", "steps.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + sources()
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if verbose or res.returncode != 0:
        print(log)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed; see paper_1811_05903_b200/build.log")
    # Post-link pass: operand-reuse hints on the FP64 instructions of the fp64 force kernels (sass_reuse.py).
    # It verifies its own output by re-disassembly and restores the library if anything but the hints changed;
    # the unpatched library is equally correct (slower), so a failure here is logged, not fatal.
    try:
        from . import sass_reuse
        n = sass_reuse.patch(LIB)
        note = f"sass_reuse: {n} instructions patched"
    except Exception as exc:  # noqa: BLE001
        note = f"sass_reuse: skipped ({exc})"
    with open(os.path.join(HERE, "build.log"), "a") as f:
        f.write("\n" + note + "\n")
    if verbose:
        print(note)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
