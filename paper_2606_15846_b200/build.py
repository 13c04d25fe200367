"""Build libflashnav.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

_DIR = os.path.dirname(os.path.abspath(__file__))
SOURCES = [os.path.join(_DIR, "csrc", f) for f in ("flashnav.cu", "fn_peaks.cu")]
HEADERS = [os.path.join(_DIR, "csrc", f) for f in ("fn_common.cuh", "fn_beam.cuh", "fn_env.cuh", "fn_features.cuh", "fn_fixed_step.cuh", "fn_reset_beam.cuh", "fn_step_split.cuh")] + \
          [os.path.join(os.path.dirname(_DIR), "include", "flashnav.h")]
LIB = os.path.join(_DIR, "libflashnav.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
