"""CPU-only checks of the C-ABI library: it loads without a GPU, exports every symbol that
include/lbm.h declares, validates arguments before touching CUDA, and documents a lattice order
identical to the oracle's (each side wrote its own table)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import lattice as oracle_lattice
from paper_2201_11330_b200 import build as lbm_build
from paper_2201_11330_b200 import lbm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    lbm_build.build()
    return lbm.load()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "lbm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = _declared_functions()
    assert set(names) == set(lbm.SYMBOLS), (names, lbm.SYMBOLS)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/lbm.h but not exported"
        assert getattr(lib, n).argtypes is not None, f"{n}: the binding sets no argtypes (pointers would be truncated)"


def test_signatures_have_no_torch_types():
    src = open(os.path.join(ROOT, "include", "lbm.h")).read()
    assert 'extern "C"' in src
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    assert "torch" not in code.lower() and "at::" not in code and "#include <stdint.h>" in code


def test_d2q9_table_is_the_papers_eq3_eq4(lib):
    """The library's D2Q9 table against the values the paper prints (tests/golden/d2q9_eq3_eq4.txt)."""
    from fractions import Fraction
    rows = {}
    with open(os.path.join(ROOT, "tests", "golden", "d2q9_eq3_eq4.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, *v = line.split()
                rows[k] = v
    e, t = lbm.lbm_lattice(lbm.LBM_D2Q9)
    assert e[:, 0].tolist() == [int(v) for v in rows["ex"]]
    assert e[:, 1].tolist() == [int(v) for v in rows["ey"]]
    assert (e[:, 2] == 0).all()
    assert t.tolist() == [float(Fraction(v)) for v in rows["t"]]


@pytest.mark.parametrize("Q", [9, 19, 27])
def test_lattice_order_matches_oracle(lib, Q):
    e, t = lbm.lbm_lattice(Q)
    eo, to = oracle_lattice(Q)
    assert (e == eo).all()
    assert (t == to).all()


def test_invalid_arguments_fail_before_cuda(lib):
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create(8, 8, 8, 19, 0.5)  # tau <= 0.5
    assert "tau" in lbm.lbm_last_error()
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create(8, 8, 8, 15, 0.8)  # unknown lattice
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create(0, 8, 8, 19, 0.8)
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create(8, 8, 8, 19, 0.8, lbm.make_bc(face_kind=[1, 0, 0, 0, 0, 0]))  # unpaired periodic
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create(8, 8, 8, 19, 0.8, lbm.make_bc(face_kind=[7, 7, 0, 0, 0, 0]))
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create(8, 8, 8, 19 | (3 << 12), 0.8)  # unknown scheme
    assert lib.lbm_step(None, 1) == lbm.LBM_EINVAL
    assert lib.lbm_init_equilibrium(None, None, None) == lbm.LBM_EINVAL
    assert lib.lbm_moments(None, None, None, None) == lbm.LBM_EINVAL
    assert lib.lbm_time(None) == -1
    lib.lbm_destroy(None)  # no-op
    assert lbm.lbm_lattice(19)[0].shape == (19, 3)
    e = (C.c_int32 * 3)()
    assert lib.lbm_lattice(5, e, (C.c_double * 1)()) == lbm.LBM_EINVAL


def test_size_limits_are_checked_before_cuda(lib):
    """Cell indices are 32-bit: nx*ny*nz >= 2^31 is refused (LBM_EUNSUPPORTED) before any CUDA call.  In-plane storage
    offsets are 32-bit too, but a plane with Q*nx*ny >= 2^31 (D2Q9 16384^2) is NOT refused: it is stored as a plain
    structure of arrays (include/lbm.h LBM_LAYOUT_ROWS; the GPU test test_large_plane_beyond_32bit_row_offsets_equals_its_tile
    runs it) — without a device the call gets as far as the allocation and fails there."""
    with pytest.raises(lbm.LBMError) as ei:
        lbm.lbm_create(2048, 1024, 1024, 19, 0.8)
    assert ei.value.code == lbm.LBM_EUNSUPPORTED or "2^31" in str(ei.value)
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(lbm.LBMError) as ei:
            lbm.lbm_create(16384, 16384, 1, 9, 0.8)
        assert "2^31" not in str(ei.value) and "must be" not in str(ei.value)  # an allocation / CUDA error, not a refusal
    assert lib.lbm_debug_arm(None, 1) == lbm.LBM_EINVAL
    assert lib.lbm_debug_check(None) == lbm.LBM_EINVAL


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(lbm, "_lib", None)
    monkeypatch.setattr(lbm, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        lbm.load()


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2201_11330_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), fn
                assert "lbm_oracle" not in txt, fn
    otxt = open(os.path.join(ROOT, "oracle", "lbm_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "binding.py")).read()
    assert "paper_2201_11330_b200" not in re.sub(r"//.*|#.*", "", otxt)
    assert "lbm_kernels" not in re.sub(r"//.*", "", otxt)
