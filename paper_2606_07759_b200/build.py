"""Build step: compile the C-ABI library ``libsynim.so`` in-tree with nvcc for sm_100a.

``python -m paper_2606_07759_b200.build`` (or ``__graft_entry__.build()``) cross-compiles without a
GPU.  The library links the static CUDA runtime only, so it loads on a box without a driver (the
compute entry points then return an error; there is no CPU fallback).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsynim.so")
SOURCES = ("synim_api.cu", "synim_kernels.cu", "synim_strip.cu", "synim_popt.cu")
HEADERS = ("synim_device.h", os.path.join("..", "..", "include", "synim.h"))

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-O2,-Wall", "--shared", "-cudart", "static", "-ldl"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA extension cannot be built")
    return exe


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False, extra=(), out: str = LIB) -> str:
    """Compile csrc/*.cu into paper_2606_07759_b200/libsynim.so (or ``out``); returns its path.
    ``extra=("-DSYNIM_CHECKS",)`` gives the debug build whose kernels trap on any shared-memory, weight-map
    or slope-table access outside its bounds."""
    if out == LIB and not force and not stale():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-o", out] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.check_call(cmd)
    return out


if __name__ == "__main__":
    print(build_library(force=True, verbose="-v" in sys.argv))
