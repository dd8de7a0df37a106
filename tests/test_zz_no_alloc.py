"""lbm_diagnostics_static: the Monitor reduction for callers that are not allowed to allocate device memory.

Who that is: a process whose GPU memory is owned by a pool of its own (torch's caching allocator, a solver that
sizes its arrays to the card) and where a cudaMalloc behind the pool's back fails or takes the room of the next
time step; a monitor inside a running time loop, which the device-wide synchronisation of cudaMalloc / cudaFree
would stall; code that holds only a pointer to somebody else's populations and no handle (lbm_create allocates).
For them the library keeps the scratch of the reduction in a fixed 2 MiB array of its own, which is why grids beyond
LBM_STATIC_MAX_CELLS are refused and why every call on a device shares (and inherits) the same scratch.

What is checked here: the result equals what the handle-based path (lbm_set_populations + lbm_moments) gives on the
same populations, within the tolerances tests/test_gpu_parity.py uses for the diagnostics (sums 1e-12, max / min
1e-14, the non-finite count exactly) — on calls made back to back, the second one smaller than the first so that it
runs over records the first call left behind; that free device memory does not move across a call; and that sizes
beyond the limit are refused with a message that names the limit.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure in this
add-on must not hide the parity tests.  It passes alone in a fresh process (its first call then does the per-device
set-up) and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def lbm():
    from paper_2201_11330_b200 import build as lbm_build
    from paper_2201_11330_b200 import lbm as _lbm
    lbm_build.build()
    _lbm.load()  # raises loudly if the CUDA library is missing
    return _lbm


def populations(Q, N, seed, amp=0.2):
    """Seeded non-equilibrium populations around 1/Q (no LBM arithmetic: any positive values do)."""
    rng = np.random.default_rng(seed)
    return (1.0 / Q) * (1.0 + amp * rng.uniform(-1.0, 1.0, (Q, N)))


def existing_path(lbm, dims, Q, eq, force, f_dev):
    """The 8 diagnostics through a handle: lbm_set_populations + lbm_moments (scratch from cudaMalloc)."""
    s = lbm.Solver(*dims, Q, 0.8, eq=eq, force=force)
    s.set_populations(f_dev)
    d = s.diagnostics()
    s.close()
    return d


def assert_same(d_new, d_ref):
    np.testing.assert_allclose(d_new[:5], d_ref[:5], rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(d_new[5:7], d_ref[5:7], rtol=1e-14)
    assert d_new[7] == d_ref[7]


# ------------------------------------------------------------------------------------------ no GPU needed

def test_sizes_beyond_the_fixed_scratch_are_refused(lbm):
    """Argument checks come before any CUDA call, so this runs on a box without a GPU too."""
    lib = lbm.load()
    fake = C.c_void_p(256)  # never dereferenced: the call must fail on the size first
    rc = lib.lbm_diagnostics_static(fake, lbm.LBM_STATIC_MAX_CELLS + 1, lbm.LBM_D3Q19, None, fake, None)
    assert rc == lbm.LBM_EINVAL
    msg = lbm.lbm_last_error()
    assert "LBM_STATIC_MAX_CELLS" in msg and str(lbm.LBM_STATIC_MAX_CELLS) in msg, msg
    assert lib.lbm_diagnostics_static(fake, 0, lbm.LBM_D3Q19, None, fake, None) == lbm.LBM_EINVAL
    assert lib.lbm_diagnostics_static(fake, 64, 15, None, fake, None) == lbm.LBM_EINVAL  # no such lattice
    assert lib.lbm_diagnostics_static(fake, 64, lbm.LBM_D3Q19 | lbm.LBM_STORE_F32, None, fake, None) == lbm.LBM_EINVAL
    assert lib.lbm_diagnostics_static(None, 64, lbm.LBM_D3Q19, None, fake, None) == lbm.LBM_EINVAL
    assert lib.lbm_diagnostics_static(fake, 64, lbm.LBM_D3Q19, None, None, None) == lbm.LBM_EINVAL


# ------------------------------------------------------------------------------------------ on the B200

CASES = [
    # Q, equilibrium flag name, body force, first grid (several 4096-cell blocks + a ragged tail), second grid (part of one block)
    (19, "LBM_EQ_STANDARD", None, (37, 21, 19), (16, 12, 10)),
    (19, "LBM_EQ_INCOMP", (1e-3, -2e-3, 5e-4), (37, 21, 19), (16, 12, 10)),
    (27, "LBM_EQ_STANDARD", (1e-3, -2e-3, 5e-4), (33, 17, 23), (9, 7, 5)),
    (27, "LBM_EQ_INCOMP", None, (33, 17, 23), (9, 7, 5)),
    (9, "LBM_EQ_STANDARD", (2e-3, 1e-3, 0.0), (131, 67, 3), (40, 30, 1)),
]


@pytest.mark.gpu
@pytest.mark.parametrize("Q,eqname,force,dims1,dims2", CASES)
def test_two_calls_in_a_row_match_the_handle_path(lbm, Q, eqname, force, dims1, dims2):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    eq = getattr(lbm, eqname)
    stream = torch.cuda.current_stream().cuda_stream
    out = torch.empty(8, dtype=torch.float64, device="cuda")  # the caller's output buffer, reused by every call

    n1, n2 = int(np.prod(dims1)), int(np.prod(dims2))
    f1 = populations(Q, n1, seed=11 * Q)
    f2 = populations(Q, n2, seed=13 * Q, amp=0.35)
    f2[Q // 2, 5] = np.nan          # two non-finite cells: counted in [7], left out of the sums
    f2[1, n2 - 1] = np.inf
    f1_dev = torch.from_numpy(f1.reshape(-1)).cuda()
    f2_dev = torch.from_numpy(f2.reshape(-1)).cuda()
    ref1 = existing_path(lbm, dims1, Q, eq, force, f1_dev)
    ref2 = existing_path(lbm, dims2, Q, eq, force, f2_dev)
    assert ref2[7] == 2

    # call 1 (in a fresh process this is also the per-device set-up)
    lbm.lbm_diagnostics_static(f1_dev, Q | eq, out, force=force, stream=stream)
    torch.cuda.synchronize()
    d1 = out.cpu().numpy().copy()
    assert_same(d1, ref1)

    # call 2, straight after, on a smaller grid: the scratch still holds call 1's records beyond the first one
    free_before = torch.cuda.mem_get_info()[0]
    lbm.lbm_diagnostics_static(f2_dev, Q | eq, out, force=force, stream=stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "free device memory moved across a call that must not allocate"
    d2 = out.cpu().numpy().copy()
    assert_same(d2, ref2)

    # and the first input again: fixed 4096-cell records and a fixed folding order => the same bits as call 1
    lbm.lbm_diagnostics_static(f1_dev, Q | eq, out, force=force, stream=stream)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == d1).all()


@pytest.mark.gpu
def test_largest_accepted_grid_matches_the_handle_path(lbm):
    """ncells = LBM_STATIC_MAX_CELLS exactly (every record of the fixed array in use), D2Q9 to keep it at 9.7 GB."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    Q, dims = 9, (8192, 16384, 1)
    n = dims[0] * dims[1]
    assert n == lbm.LBM_STATIC_MAX_CELLS
    if torch.cuda.mem_get_info()[0] < 40 * (1 << 30):
        pytest.skip("needs 40 GB of free device memory (input + the handle's two buffers)")
    g = torch.Generator(device="cuda")
    g.manual_seed(2201_11330)
    f_dev = (1.0 / Q) * (1.0 + 0.2 * (2.0 * torch.rand(Q * n, dtype=torch.float64, device="cuda", generator=g) - 1.0))
    ref = existing_path(lbm, dims, Q, lbm.LBM_EQ_STANDARD, None, f_dev)
    out = torch.empty(8, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    for _ in range(2):  # two calls in a row
        out.fill_(-1.0)
        lbm.lbm_diagnostics_static(f_dev, Q, out, stream=stream)
        torch.cuda.synchronize()
        assert_same(out.cpu().numpy(), ref)
