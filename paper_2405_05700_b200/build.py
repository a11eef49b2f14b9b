"""Builds the CUDA library in-tree: ``python -m paper_2405_05700_b200.build``.

nvcc cross-compiles for sm_100a without a GPU; the resulting ``libpp.so`` sits next to this file
(git-ignored, but it travels to the GPU box with the repo snapshot).

Developer knob: the environment variable ``PP_NVCC_EXTRA`` is appended to the nvcc command line (e.g.
``-DPP_MIN_BLOCKS=3`` for an occupancy experiment).  It is part of the hash ``bench.py`` stores with the measured
instructions per flight, so a library built with extra flags never borrows the roofline constant of the default
build.  The product build uses none.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpp.so")
SOURCES = ["pp_kernels.cu", "pp_api.cpp", "pp_ipc.cpp", "pp_multi.cpp"]
DEPS = SOURCES + ["pp_device.cuh", "pp_guard.cuh", "pp_types.h", "pp_internal.h", os.path.join("..", "..", "include", "pp.h"),
                  os.path.join("..", "..", "include", "pp_ipc.h"), os.path.join("..", "..", "include", "pp_multi.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build(force: bool = False, verbose: bool = False, out: str = LIB, defines=()) -> str:
    """Builds libpp.so (or, for the tests, a variant of it: `out` elsewhere, with extra -D `defines`)."""
    deps = [os.path.join(CSRC, d) for d in DEPS]
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(d) for d in deps):
        return out
    extra = os.environ.get("PP_NVCC_EXTRA", "").split()  # e.g. -DPP_MIN_BLOCKS=4 (tuning experiments)
    cmd = [nvcc()] + NVCC_FLAGS + extra + ["-D" + d for d in defines] + (["-Xptxas", "-v"] if verbose else []) + \
        ["-o", out] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lrt", "-lpthread"]
    subprocess.check_call(cmd)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
