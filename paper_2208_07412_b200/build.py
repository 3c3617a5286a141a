"""Build libtpcca.so IN-TREE with nvcc for sm_100a.  Usage: python -m paper_2208_07412_b200.build [--force]

Flags are part of the arithmetic contract: --fmad=false (no FMA contraction),
nvcc's defaults -prec-div=true -prec-sqrt=true -ftz=false (IEEE division / sqrt, denormals kept).
nvcc cross-compiles without a GPU, so this also is the "does it build" check.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtpcca.so")
SOURCES = ["tpcca_api.cu", "tpcca_noalloc.cu"]
DEPS = ["tpcca_api.cu", "tpcca_noalloc.cu", "tpcca_pipeline.cuh", "tpcca_dev.cuh", "k_grid.cuh", "k_links.cuh", "k_tracklets.cuh", "k_select.cuh", "k_merge.cuh"]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "--fmad=false", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libtpcca.so cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, d) for d in DEPS] + [os.path.join(ROOT, "include", "tpcca.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, "-I", os.path.join(ROOT, "include")]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
