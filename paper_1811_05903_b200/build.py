"""Build the C-ABI library in-tree: nvcc (sm_100a only) -> paper_1811_05903_b200/libsteps_b200.so.

Usage: python -m paper_1811_05903_b200.build [--force] [--verbose] [--unpatched]
nvcc cross-compiles without a GPU; the built .so travels to the GPU box with the snapshot.

After linking, sass_reuse.py adds operand-reuse hints to the FP64 / packed-fp32 instructions of the force kernels
(worth ~3.5 % on the fp64 kernels).  The pass is part of the build: if it cannot be applied (a new
toolkit whose encoding fails the calibration, cuobjdump missing) the build FAILS instead of silently shipping the slower
library.  STEPS_NO_SASS_PATCH=1 in the environment skips it on purpose.  What was done is recorded beside the library in
libsteps_b200.so.buildinfo (JSON; steps.build_info() reads it, bench.py prints it).  `--unpatched` / build_unpatched()
builds libsteps_b200_unpatched.so from the same sources without the pass, for the A/B test that the hints do not
change results (tests/test_parity_gpu.py::test_sass_reuse_patch_is_bit_identical)."""
from __future__ import annotations

import glob
import json
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsteps_b200.so")
LIB_UNPATCHED = os.path.join(HERE, "libsteps_b200_unpatched.so")

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
        os.path.join(os.path.dirname(HERE), "include", "steps.h"), os.path.join(HERE, "sass_reuse.py")]


def _fresh(lib: str) -> bool:
    return os.path.exists(lib) and os.path.exists(lib + ".buildinfo") and all(
        os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps())


def _compile(lib: str, verbose: bool) -> list[str]:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", lib] + sources()
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    if lib == LIB:
        with open(os.path.join(HERE, "build.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + log)
    if verbose or res.returncode != 0:
        print(log)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed; see paper_1811_05903_b200/build.log")
    return cmd


def _write_info(lib: str, cmd: list[str], patched: int | None, note: str) -> None:
    with open(lib + ".buildinfo", "w") as f:
        json.dump({"nvcc": " ".join(cmd), "sass_reuse_patched_instructions": patched, "sass_reuse": note}, f)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and _fresh(LIB):
        return LIB
    cmd = _compile(LIB, verbose)
    if os.environ.get("STEPS_NO_SASS_PATCH") == "1":
        _write_info(LIB, cmd, None, "skipped on request (STEPS_NO_SASS_PATCH=1)")
        return LIB
    from . import sass_reuse
    try:
        n = sass_reuse.patch(LIB)
    except Exception as exc:
        os.remove(LIB)                      # never leave an unpatched library that looks like the product
        raise RuntimeError(f"sass_reuse could not be applied ({exc}); fix it or build with STEPS_NO_SASS_PATCH=1") from exc
    if n == 0:
        os.remove(LIB)
        raise RuntimeError("sass_reuse found nothing to patch: the force kernels' names or SASS changed")
    _write_info(LIB, cmd, n, "applied")
    with open(os.path.join(HERE, "build.log"), "a") as f:
        f.write(f"\nsass_reuse: {n} instructions patched\n")
    if verbose:
        print(f"sass_reuse: {n} instructions patched")
    return LIB


def build_unpatched(force: bool = False, verbose: bool = False) -> str:
    """The same sources and flags without the post-link pass (A/B test only; nothing in the product loads it)."""
    if not force and _fresh(LIB_UNPATCHED):
        return LIB_UNPATCHED
    cmd = _compile(LIB_UNPATCHED, verbose)
    _write_info(LIB_UNPATCHED, cmd, None, "not applied (A/B build)")
    return LIB_UNPATCHED


def build_info(lib: str = LIB) -> dict:
    try:
        with open(lib + ".buildinfo") as f:
            return json.load(f)
    except (OSError, ValueError):
        return {"sass_reuse": "unknown (no buildinfo beside the library)", "sass_reuse_patched_instructions": None}


if __name__ == "__main__":
    if "--unpatched" in sys.argv:
        print(build_unpatched(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
