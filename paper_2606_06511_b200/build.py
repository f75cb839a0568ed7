"""Builds paper_2606_06511_b200/libtt.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
SRC = HERE / "csrc" / "tt_lib.cu"
DEPS = [SRC, HERE / "csrc" / "tt_kernels.cuh", HERE / "csrc" / "tt_geom.cuh", HERE / "csrc" / "tt_probe.cuh", HERE / "csrc" / "tt_broad.cuh", HERE / "csrc" / "tt_solve.cuh", HERE / "csrc" / "tt_exact.cuh", HERE / "csrc" / "tt_membrane.cuh", HERE.parent / "include" / "tt.h"]
LIB = HERE / "libtt.so"

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr"]


def nvcc_path() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and LIB.exists() and all(LIB.stat().st_mtime >= d.stat().st_mtime for d in DEPS):
        return LIB
    cmd = [nvcc_path(), *NVCC_FLAGS, str(SRC), "-o", str(LIB)]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    return LIB


PROFILE_LIB = HERE / "libtt_prof.so"


def build_profile() -> Path:
    """A second library with the phase timers of K4 compiled in (-DTT_K4_PROFILE: clock64() marks summed per phase,
    read through tt_debug_k4_prof).  A profiling build: `bench.py --k4-phases` loads it; nothing else does."""
    if PROFILE_LIB.exists() and all(PROFILE_LIB.stat().st_mtime >= d.stat().st_mtime for d in DEPS):
        return PROFILE_LIB
    subprocess.run([nvcc_path(), *NVCC_FLAGS, "-DTT_K4_PROFILE", str(SRC), "-o", str(PROFILE_LIB)], check=True)
    return PROFILE_LIB


if __name__ == "__main__":
    if "--profile" in sys.argv:
        print(build_profile())
    else:
        build(force="--force" in sys.argv, verbose="-v" in sys.argv)
        print(LIB)
