"""Build the CUDA library (csrc/*.cu -> paper_2201_11330_b200/liblbm_b200.so) for sm_100a.

`python -m paper_2201_11330_b200.build [--force] [--verbose] [--ptxas]`.  nvcc cross-compiles
without a GPU.  The kernel instantiations (csrc/lbm_inst.cu) are compiled once per lattice and
part into separate objects, in parallel, then linked with the C ABI (csrc/lbm_abi.cu, csrc/lbm_static.cu).  The .so
is built in-tree (git-ignored) so that it travels to the GPU box with the repo.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblbm_b200.so")
DEPS = ["lbm_abi.cu", "lbm_inst.cu", "lbm_static.cu", "lbm_kernels.cuh", "lbm_launch.cuh", os.path.join(ROOT, "include", "lbm.h")]
LATTICES = (9, 19, 27)
PARTS = (0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10)  # A/B step, AA even, AA odd, export/import/init/geometry, moments/force, A/B slab step,
                                  # A/B step with SYMMETRY faces, A/B slab step with SYMMETRY faces, persistent A/B kernel, persistent AA kernel,
                                  # A/B two steps per pass

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo", "--fmad=true",
    "-Xcompiler", "-fPIC", "-diag-suppress", "177",
    "-Xfatbin", "-compress-all",  # 145 MB -> 36 MB of device code (the .so travels to the GPU box with every call)
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


def _units():
    """(object path, source, extra defines) of every translation unit."""
    units = [(os.path.join(OBJ, "lbm_abi.o"), os.path.join(CSRC, "lbm_abi.cu"), []),
             (os.path.join(OBJ, "lbm_static.o"), os.path.join(CSRC, "lbm_static.cu"), [])]  # lbm_diagnostics_static
    for q in LATTICES:
        for part in PARTS:
            units.append((os.path.join(OBJ, f"lbm_inst_q{q}_p{part}.o"), os.path.join(CSRC, "lbm_inst.cu"),
                          [f"-DLBM_Q={q}", f"-DLBM_PART={part}"]))
    return units


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = _nvcc()
    os.makedirs(OBJ, exist_ok=True)
    units = _units()

    def compile_one(unit):
        obj, src, defs = unit
        cmd = [nvcc, *NVCC_FLAGS, *extra, *defs, "-c", "-o", obj, src]
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        r = subprocess.run(cmd, capture_output=True, text=True)
        return unit, r

    # biggest units first (D3Q27 steps) so that the pool stays busy
    order = sorted(units, key=lambda u: (("-DLBM_Q=27" in u[2]) * 2 + ("-DLBM_Q=19" in u[2])), reverse=True)
    with cf.ThreadPoolExecutor(max_workers=max(1, min(len(units), os.cpu_count() or 1))) as pool:
        results = list(pool.map(compile_one, order))
    failed = False
    for (obj, src, defs), r in results:
        if r.returncode != 0 or (r.stderr.strip() and (verbose or extra)):
            print(f"--- nvcc {' '.join(defs)} {os.path.basename(src)}\n{r.stdout}{r.stderr}", file=sys.stderr)
        failed |= r.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed (see messages above)")
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", "-o", LIB] + [u[0] for u in units]
    if verbose:
        print(" ".join(link), file=sys.stderr)
    subprocess.run(link, check=True)
    return LIB


if __name__ == "__main__":
    args = sys.argv[1:]
    extra = (["-Xptxas", "-v"] if "--ptxas" in args else []) + [a for a in args if a.startswith("-D")]
    print(build(force="--force" in args or bool(extra), verbose=True, extra=extra))
