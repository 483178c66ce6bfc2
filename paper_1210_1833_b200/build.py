"""Build libcute_b200.so (the C-ABI library of include/cute_b200.h) in-tree with nvcc for sm_100a.

    python -m paper_1210_1833_b200.build [--force]

nvcc cross-compiles without a GPU.  The library is linked against the static CUDA runtime so
that it loads by itself (ctypes) next to PyTorch.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcute_b200.so")
SOURCES = ["cute_api.cu", "grid_build.cu", "pair_count.cu", "pair_kind_monopole.cu", "pair_kind_angular.cu",
           "pair_kind_rmu.cu", "pair_kind_radial.cu", "pair_kind_pisigma.cu", "density_grid.cu", "peaks.cu", "no_alloc.cu"]
HEADERS = [os.path.join(CSRC, "cute_internal.h"), os.path.join(CSRC, "pair_kernel.cuh"),
           os.path.join(HERE, "..", "include", "cute_b200.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]
if os.environ.get("CUTE_MAX_WARPS"):          # experiments only: warps per CTA (default 16, cute_internal.h)
    NVCC_FLAGS += ["-DCUTE_MAX_WARPS=" + os.environ["CUTE_MAX_WARPS"]]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        objs.append(o)
        cmd = [_nvcc(), *NVCC_FLAGS, "-c", os.path.join(CSRC, s), "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [_nvcc(), "-shared", "-o", LIB, *objs, "-cudart", "static"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
