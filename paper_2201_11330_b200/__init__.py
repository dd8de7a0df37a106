"""B200-native fused stream-collide lattice-Boltzmann hot path (IMEXLBM, arXiv 2201.11330).

`paper_2201_11330_b200.lbm` is the thin ctypes binding over the C-ABI library declared in
include/lbm.h (built from csrc/ by `python -m paper_2201_11330_b200.build`); it is loaded
lazily on first use and fails loudly if the CUDA library is missing — there is no CPU path.
`paper_2201_11330_b200.inputs` holds the seeded synthetic workloads (numpy only).
"""
__all__ = ["inputs", "lbm", "build"]
