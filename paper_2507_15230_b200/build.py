"""Build step: nvcc -> paper_2507_15230_b200/csrc/libgale.so (sm_100a only, in-tree)."""
from __future__ import annotations

import os
import subprocess

CSRC = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc")
LIB = os.path.join(CSRC, "libgale.so")
LIB_CHECKED = os.path.join(CSRC, "libgale_checked.so")   # -DGALE_CHECK_BOUNDS=1 (tests/test_gpu_bounds.py)
SOURCES = ["gale_lib.cu"]
DEPS = SOURCES + ["gale_kernels.cuh", "gale_walk.cuh", "gale_init.cuh", "gale_sub.cuh", "gale_canon.cuh", os.path.join("..", "..", "include", "gale.h")]

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "170"]


def is_stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build_library(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """Compile the CUDA library if it is missing or older than its sources. `checked` builds the
    bounds-checked variant (same sources, -DGALE_CHECK_BOUNDS=1) next to it."""
    lib = LIB_CHECKED if checked else LIB
    if force or is_stale(lib):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = lib + f".{os.getpid()}.tmp"
        cmd = ([nvcc] + NVCC_FLAGS + (["-DGALE_CHECK_BOUNDS=1"] if checked else []) +
               (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES)
        subprocess.check_call(cmd, cwd=CSRC)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
