"""Build the CUDA library (csrc/*.cu -> paper_2201_11330_b200/liblbm_b200.so) for sm_100a.

`python -m paper_2201_11330_b200.build [--force] [--verbose]`.  nvcc cross-compiles without a
GPU.  The .so is built in-tree (git-ignored) so that it travels to the GPU box with the repo.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblbm_b200.so")
SOURCES = ["lbm_abi.cu"]
DEPS = ["lbm_abi.cu", "lbm_kernels.cuh", os.path.join(ROOT, "include", "lbm.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "--fmad=true",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-diag-suppress", "177",
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for d in DEPS:
        p = d if os.path.isabs(d) else os.path.join(CSRC, d)
        if os.path.getmtime(p) > t:
            return True
    return False


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    args = sys.argv[1:]
    extra = ["-Xptxas", "-v"] if "--ptxas" in args else []
    print(build(force="--force" in args or bool(extra), verbose=True, extra=extra))
