"""Build libsnaps.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libsnaps.so")
SOURCES = ["api.cu", "knn_lattice.cu", "range_lattice.cu", "misc_kernels.cu", "pivot_sort.cu", "ranking.cu", "range_grid.cu", "eps_search.cu"]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    # no implicit mul+add contraction: the kernels place their FMAs explicitly so that the
    # main loop and the rare paths round identically
    "-fmad=false",
    "-Xcompiler", "-fPIC", "-shared",
    "-diag-suppress", "177",   # phase-clock variables that only the developer stats build reads
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "snaps.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + f".{os.getpid()}.tmp"
        extra = os.environ.get("SNAPS_NVCC_EXTRA", "").split()   # developer builds, e.g. -DSNAPS_STATS
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-o", tmp, *[os.path.join(CSRC, s) for s in SOURCES]]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
