"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances (BASELINE.json north_star): max |df| <= 1e-12 for fp64
storage, <= 2e-5 relative for the fp32-storage variant.  Run with `pytest -m gpu` on a B200.
"""
import dataclasses

import numpy as np
import pytest

from oracle import Oracle
from oracle.binding import EQ_INCOMP, EQ_STANDARD
from paper_2201_11330_b200 import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
TOL = 1e-12

B, M, P = inputs.FACE_BOUNCE, inputs.FACE_MOVING, inputs.FACE_PERIODIC


@pytest.fixture(scope="module")
def lbm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_11330_b200 import lbm as _lbm
    _lbm.load()  # raises loudly if the CUDA library is missing
    return _lbm


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def eq_flag(lbm, eq):
    return lbm.LBM_EQ_INCOMP if eq == EQ_INCOMP else lbm.LBM_EQ_STANDARD


def make_pair(lbm, dims, Q, tau, eq=EQ_STANDARD, scheme=None, face_kind=None, face_u=None, force=None, store=0):
    nx, ny, nz = dims
    o = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=face_kind, face_u=face_u, force=force)
    s = lbm.Solver(nx, ny, nz, Q, tau, eq=eq_flag(lbm, eq), scheme=scheme or lbm.LBM_SCHEME_AB, store=store,
                   face_kind=face_kind, face_u=face_u, force=force)
    return o, s


def random_f(Q, N, seed, amp=0.2):
    """Random non-equilibrium populations around the weights (from the oracle-independent lattice rule:
    weights only matter as a positive scale here)."""
    rng = np.random.default_rng(seed)
    base = np.full((Q, 1), 1.0 / Q)
    return base * (1.0 + amp * rng.uniform(-1, 1, (Q, N)))


def schemes(lbm):
    return [("ab", lbm.LBM_SCHEME_AB), ("aa", lbm.LBM_SCHEME_AA)]


FACE_CASES = {
    "periodic": ([P] * 6, None),
    "channel_z": ([P, P, P, P, B, B], None),
    "couette_z": ([P, P, P, P, B, M], {5: (0.05, 0.02, 0.0)}),
    "cavity": ([B, B, B, B, B, M], {5: (0.1, 0.0, 0.0)}),
    "mixed": ([B, M, P, P, M, B], {1: (0.0, 0.03, -0.02), 4: (0.05, 0.01, 0.0)}),
    "all_moving": ([M] * 6, {k: (0.01 * (k + 1), -0.02, 0.005 * k) for k in range(6)}),
}
# open faces (D:R22: velocity inlet, pressure outlet at the default density 1) for the two-step kernel's tests
PR = inputs.FACE_PRESSURE
OPEN_CASES = {
    "inlet_outlet_x": ([M, PR, B, B, P, P], {0: (0.04, 0.0, 0.0)}),
    "inlet_outlet_z": ([P, P, P, P, M, PR], {4: (0.0, 0.01, 0.03)}),
}
FACE_CASES_TWO_STEP = dict(FACE_CASES, **OPEN_CASES)


def face_u_of(spec):
    fu = np.zeros((6, 3))
    for k, v in (spec or {}).items():
        fu[k] = v
    return fu


# --------------------------------------------------------------------------- element-wise parity, all variants

@pytest.mark.parametrize("scheme", ["ab", "aa"])
@pytest.mark.parametrize("faces", list(FACE_CASES))
@pytest.mark.parametrize("Q,eq,forced", [(19, EQ_STANDARD, False), (19, EQ_STANDARD, True), (19, EQ_INCOMP, False),
                                         (19, EQ_INCOMP, True), (27, EQ_STANDARD, False), (27, EQ_STANDARD, True),
                                         (27, EQ_INCOMP, True), (9, EQ_STANDARD, False), (9, EQ_INCOMP, True)])
def test_random_populations_ragged_grid(lbm, scheme, faces, Q, eq, forced):
    """Ragged 37x21x13 grid (several 32-wide tiles + a tail in x, odd y and z), random non-equilibrium
    populations, 7 steps (odd: the AA scheme is compared in its swapped phase too)."""
    dims = (37, 21, 13)
    N = dims[0] * dims[1] * dims[2]
    fk, fu = FACE_CASES[faces]
    fu = face_u_of(fu)
    F = (2e-4, -1e-4, 3e-4) if forced else None
    if Q == 9:
        # D2Q9 has no z-links: z faces must be periodic for the comparison to mean anything, and MOVING z faces
        # would never be crossed.  Keep the x / y face kinds of the case.
        fk = list(fk[:4]) + [P, P]
    o, s = make_pair(lbm, dims, Q, 0.77, eq, dict(schemes(lbm))[scheme], fk, fu, F)
    f0 = random_f(Q, N, seed=Q + 100 * eq)
    o.set_f(f0)
    s.set_populations(dev(f0))
    assert np.abs(s.get_populations().cpu().numpy() - f0).max() == 0.0  # import/export round trip is exact
    for nsteps in (1, 2, 4):  # compare after 1, 3 and 7 steps
        o.step(nsteps)
        s.step(nsteps)
        got = s.get_populations().cpu().numpy()
        assert np.abs(got - o.get_f()).max() <= TOL
    rho, u, d = s.moments()
    ro, uo, do = o.moments()
    assert np.abs(rho.cpu().numpy() - ro).max() <= 1e-13
    assert np.abs(u.cpu().numpy() - uo).max() <= 1e-13
    np.testing.assert_allclose(d[:5], do[:5], rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(d[5:7], do[5:7], rtol=1e-14)
    assert d[7] == do[7] == 0
    s.close()


@pytest.mark.parametrize("dims", [(1, 1, 1), (2, 3, 1), (4, 4, 4), (3, 2, 5), (300, 5, 3), (64, 64, 2), (33, 1, 7)])
@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_degenerate_and_edge_sizes(lbm, dims, scheme):
    """Smallest grids (wrap onto itself), a row longer than one 256-thread block, single-plane grids."""
    N = dims[0] * dims[1] * dims[2]
    for fk, fu in (([P] * 6, None), ([B, B, B, B, B, M], {5: (0.1, 0.0, 0.0)})):
        o, s = make_pair(lbm, dims, 19, 0.6, EQ_STANDARD, dict(schemes(lbm))[scheme], fk, face_u_of(fu), (1e-5, 0, 2e-5))
        f0 = random_f(19, N, seed=N)
        o.set_f(f0)
        s.set_populations(dev(f0))
        o.step(5)
        s.step(5)
        assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
        s.close()


@pytest.mark.parametrize("bx,by", [(32, 1), (32, 8), (64, 4), (128, 2), (256, 1), (32, 4)])
def test_block_shapes_give_identical_results(lbm, bx, by):
    dims = (70, 19, 6)
    N = dims[0] * dims[1] * dims[2]
    f0 = random_f(19, N, seed=5)
    ref = None
    for shape in ((0, 0), (bx, by)):
        s = lbm.Solver(*dims, 19, 0.7)
        s.set_block(*shape)
        s.set_populations(dev(f0))
        s.step(3)
        got = s.get_populations().cpu().numpy()
        s.close()
        if ref is None:
            ref = got
        else:
            assert (got == ref).all()


# --------------------------------------------------------------------------- init, moments, host variants

@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_STANDARD), (19, EQ_INCOMP)])
@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_init_equilibrium_matches_oracle(lbm, Q, eq, scheme):
    dims = (20, 9, 11)
    N = dims[0] * dims[1] * dims[2]
    rng = np.random.default_rng(11)
    rho = 1 + 0.05 * rng.standard_normal(N)
    u = 0.05 * rng.standard_normal((3, N))
    fk, fu = FACE_CASES["cavity"]
    o, s = make_pair(lbm, dims, Q, 0.8, eq, dict(schemes(lbm))[scheme], fk, face_u_of(fu))
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= 1e-15
    assert s.time == 0
    # NULL fields: rho = 1, u = 0
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= 1e-16
    s.close()


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_host_entry_points_equal_device_ones(lbm, scheme):
    w = inputs.config(0).scaled(24, steps=9)
    rho, u = w.fields()
    a = lbm.Solver.from_workload(w, scheme=dict(schemes(lbm))[scheme])
    b = lbm.Solver.from_workload(w, scheme=dict(schemes(lbm))[scheme])
    a.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    rho_h = torch.from_numpy(rho).pin_memory()
    u_h = torch.from_numpy(u.reshape(-1).copy()).pin_memory()
    b.init_equilibrium_host(rho_h, u_h)
    a.step(w.steps)
    b.step(w.steps)
    assert (a.get_populations() == b.get_populations()).all()
    ra, ua, da = a.moments()
    rb = torch.empty(w.N, dtype=torch.float64).pin_memory()
    ub = torch.empty(3 * w.N, dtype=torch.float64).pin_memory()
    db = lbm.lbm_moments_host(b.h, rb, ub, True)
    assert (ra.cpu() == rb).all() and (ua.cpu().reshape(-1) == ub).all() and (da == db).all()
    # stepping still works after the idle buffer was used as staging
    a.step(2)
    b.step(2)
    assert (a.get_populations() == b.get_populations()).all()
    a.close()
    b.close()


def test_host_arrays_may_be_reused_as_soon_as_init_returns(lbm):
    """include/lbm.h: lbm_init_equilibrium_host returns when rho / u have left the host (its copy stream is internal, so
    the caller could not wait for it).  Overwrite the pinned arrays the moment the call returns — 0.5 GB at 256^3, tens of
    milliseconds on the bus — and the initial state must still be the one made from the original values."""
    n = 256
    N = n ** 3
    g = torch.Generator(device="cuda")
    g.manual_seed(7)
    rho_d = 1.0 + 1e-3 * (torch.rand(N, dtype=torch.float64, device="cuda", generator=g) - 0.5)
    u_d = 0.05 * (torch.rand(3 * N, dtype=torch.float64, device="cuda", generator=g) - 0.5)
    rho_h = rho_d.cpu().pin_memory()
    u_h = u_d.cpu().pin_memory()
    a = lbm.Solver(n, n, n, 19, 0.6, scheme=lbm.LBM_SCHEME_AA)  # (one buffer each: 2.5 GB)
    b = lbm.Solver(n, n, n, 19, 0.6, scheme=lbm.LBM_SCHEME_AA)
    a.init_equilibrium(rho_d, u_d)
    b.init_equilibrium_host(rho_h, u_h)
    rho_h.fill_(float("nan"))  # the caller reuses its buffers at once
    u_h.fill_(float("nan"))
    fa = a.get_populations()
    a.close()
    fb = b.get_populations()
    b.close()
    assert bool(torch.isfinite(fb).all()) and torch.equal(fa, fb)


def test_nonfinite_cells_are_counted(lbm):
    dims = (8, 8, 8)
    s = lbm.Solver(*dims, 19, 0.8)
    f0 = random_f(19, 512, seed=1)
    f0[3, 17] = np.nan
    f0[5, 100] = np.inf
    s.set_populations(dev(f0))
    d = s.diagnostics()
    assert d[7] == 2 and np.isfinite(d[:7]).all()
    s.close()


def test_step_zero_and_time_counter(lbm):
    s = lbm.Solver(8, 8, 8, 19, 0.8)
    s.init_equilibrium()
    s.step(0)
    assert s.time == 0
    s.step(3)
    assert s.time == 3
    with pytest.raises(lbm.LBMError):
        s.step(-1)
    s.close()


# --------------------------------------------------------------------------- BASELINE.json configs

@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_config0_tgv32_full_length(lbm, scheme):
    """configs[0]: 32^3 periodic Taylor-Green, tau 0.8, 100 steps: parity, energy decay, conservation."""
    w = inputs.config(0)
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau)
    s = lbm.Solver.from_workload(w, scheme=dict(schemes(lbm))[scheme])
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    d0 = s.diagnostics()
    E = [d0[4]]
    for _ in range(w.steps):
        s.step(1)
        E.append(s.diagnostics()[4])
    o.step(w.steps)
    err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
    print(f"\ntest_config0_tgv32_full_length: max|df| vs oracle = {err:.2e}")
    assert err <= TOL
    d1 = s.diagnostics()
    do = o.moments(False)[2]
    np.testing.assert_allclose(d1[:5], do[:5], rtol=1e-12, atol=1e-12)
    nu, k2 = (w.tau - 0.5) / 3, 3 * (2 * np.pi / w.nx) ** 2
    slope = np.polyfit(np.arange(10, 101), np.log(E[10:101]), 1)[0]
    assert abs(slope / (-2 * nu * k2) - 1) < 0.03
    assert abs(d1[0] - d0[0]) / d0[0] < 1e-13
    np.testing.assert_allclose(d1[1:4], d0[1:4], atol=1e-11)
    s.close()


def test_config1_tgv128_full_length(lbm):
    """configs[1]: 128^3 periodic Taylor-Green, tau 0.6, 1000 steps, full-length parity against the oracle."""
    w = inputs.config(1)
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau)
    s = lbm.Solver.from_workload(w)
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    o.step(w.steps)
    s.step(w.steps)
    err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
    print(f"\ntest_config1_tgv128_full_length: max|df| vs oracle = {err:.2e}")
    assert err <= TOL
    s.close()


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_config2_cavity_analogue_full_length(lbm, scheme):
    """configs[2] on a 32^3 analogue for the full 2000 steps (the 256^3 oracle run costs 3.4e10 updates)."""
    w = inputs.config(2).scaled(32)
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, face_kind=w.face_kind, face_u=w.face_u)
    s = lbm.Solver.from_workload(w, scheme=dict(schemes(lbm))[scheme])
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    o.step(w.steps)
    s.step(w.steps)
    err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
    print(f"\ntest_config2_cavity_analogue_full_length: max|df| vs oracle = {err:.2e}")
    assert err <= TOL
    rho, u, d = s.moments()
    assert abs(d[0] - w.N) / w.N < 1e-12  # mass
    uy = u[1].cpu().numpy().reshape(32, 32, 32)
    assert np.abs(uy + uy[:, ::-1, :]).max() < 1e-13  # mirror antisymmetry
    s.close()


def test_config2_cavity256_first_steps(lbm):
    """configs[2] at its full 256^3 size, the first 200 steps ("else first 200 steps"), every
    cell against the oracle, through the kernel bench.py times for this config (stream_collide_ab2 with walls).  The
    cavity starts at rest, so the test also says how much of the box has left the rest state t_a by then (the lid's
    shear layer, and the sound waves from the two edges where the lid runs into a side wall, which travel
    c_s * 200 = 115 cells)."""
    w = inputs.config(2)
    nsteps = 200
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, face_kind=w.face_kind, face_u=w.face_u)
    s = lbm.Solver.from_workload(w)
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    rest = s.get_populations().cpu().numpy().copy()  # t_a everywhere
    l0 = s.launches
    o.step(nsteps)
    s.step(nsteps)
    assert s.launches - l0 == nsteps // 2  # two steps per launch: the walled two-step kernel took them
    got = s.get_populations().cpu().numpy()
    ref = o.get_f()
    err = float(np.abs(got - ref).max())
    moved = float((np.abs(ref - rest).max(axis=0) > 1e-12).mean())
    print(f"\ntest_config2_cavity256_first_steps: {nsteps} steps, max|df| vs oracle = {err:.2e}; "
          f"{100 * moved:.1f} % of the cells differ from the rest state by more than 1e-12")
    assert err <= TOL
    assert moved > 0.10  # the comparison is not one of fixed points
    s.close()


def test_config2_cavity_analogue_full_length_two_step_kernel(lbm):
    """configs[2]'s full 2000 steps against the oracle, every cell, through stream_collide_ab2 with walls and lid — the
    32^3 analogue above runs in the persistent kernel instead.  64 x 32 x 32 (two 32 x 8 tile columns in x, four in y)."""
    w = dataclasses.replace(inputs.config(2).scaled(32), nx=64)
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, face_kind=w.face_kind, face_u=w.face_u)
    s = lbm.Solver(w.nx, w.ny, w.nz, w.Q, w.tau, face_kind=w.face_kind, face_u=w.face_u)
    s.set_persistent(0)
    s.set_two_step(2)
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    l0 = s.launches
    o.step(w.steps)
    s.step(w.steps)
    assert w.steps == 2000 and s.launches - l0 == w.steps // 2
    err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
    print(f"\ntest_config2_cavity_analogue_full_length_two_step_kernel: max|df| vs oracle = {err:.2e}")
    assert err <= TOL
    d = s.diagnostics()
    assert abs(d[0] - w.nx * w.ny * w.nz) / (w.nx * w.ny * w.nz) < 1e-12  # mass: the lid's +- links cancel (R6)
    s.close()


def _subbox_check(lbm, w, solver, k, centers, halo=2):
    """Sampled parity at full size: f after k steps at a cell depends only on the initial fields within
    distance k, so the oracle runs on a small sub-box cut around each sample (global walls kept where the
    box touches them, cut sides are far enough away) and its core cells are compared with the GPU's."""
    Q = w.Q
    fgpu = solver.get_populations().view(Q, w.nz, w.ny, w.nx)
    n = (w.nx, w.ny, w.nz)
    worst = 0.0
    for c in centers:
        lo, hi, fk, core = [], [], list(w.face_kind), []
        for d in range(3):
            a, b = c[d] - k - halo, c[d] + k + halo + 1
            periodic = w.face_kind[2 * d] == P
            if not periodic:
                a, b = max(a, 0), min(b, n[d])
            lo.append(a)
            hi.append(b)
            # cut sides of a non-periodic axis get a resting wall (garbage confined to k cells from it)
            if not periodic:
                fk[2 * d] = w.face_kind[2 * d] if a == 0 else B
                fk[2 * d + 1] = w.face_kind[2 * d + 1] if b == n[d] else B
            cl = a + (0 if (not periodic and a == 0) else k + 1)
            ch = b - (0 if (not periodic and b == n[d]) else k + 1)
            core.append((cl, ch))
        box = tuple((lo[d], hi[d]) for d in range(3))
        rho, u = w.fields(box)
        dims = [hi[d] - lo[d] for d in range(3)]
        o = Oracle(dims[0], dims[1], dims[2], Q, w.tau, face_kind=fk, face_u=w.face_u, force=w.force)
        o.init_equilibrium(rho, u)
        o.step(k)
        fo = o.get_f().reshape(Q, dims[2], dims[1], dims[0])
        for gz in range(core[2][0], core[2][1]):
            for gy in range(core[1][0], core[1][1]):
                xs = np.arange(core[0][0], core[0][1])
                ref = fo[:, gz - lo[2], gy - lo[1], xs - lo[0]]
                got = fgpu[:, gz % n[2], gy % n[1], torch.from_numpy(xs % n[0]).cuda()].cpu().numpy()
                worst = max(worst, np.abs(got - ref).max())
    return worst


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_config3_tgv512_sampled(lbm, scheme):
    """configs[3] (headline, 512^3): sampled sub-box parity after 3 steps at corners, edges, faces and
    interior points, plus mass/momentum conservation over the steps (properties that hold at any size)."""
    w = inputs.config(3)
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w, scheme=dict(schemes(lbm))[scheme])
    rho_h = torch.from_numpy(rho).pin_memory()
    u_h = torch.from_numpy(u.reshape(-1)).pin_memory()
    s.init_equilibrium_host(rho_h, u_h)
    d0 = s.diagnostics()
    k = 3
    s.step(k)
    centers = [(0, 0, 0), (511, 511, 511), (0, 255, 511), (256, 0, 17), (100, 200, 300), (255, 256, 511), (31, 32, 33)]
    err = _subbox_check(lbm, w, s, k, centers)
    print(f"\ntest_config3_tgv512_sampled: max|df| vs oracle on the sampled sub-boxes = {err:.2e}")
    assert err <= TOL
    s.step(20 - k)
    d1 = s.diagnostics()
    assert abs(d1[0] - d0[0]) / d0[0] < 1e-13
    np.testing.assert_allclose(d1[1:4], d0[1:4], atol=1e-9)
    assert d1[7] == 0 and d1[4] < d0[4]
    s.close()


def test_config4_channel512_sampled(lbm):
    """configs[4] (D3Q27, 512^3 forced channel): sampled sub-box parity after 3 steps next to both walls and
    inside, and the plane-averaged profile against the analytic start-up series after 200 steps."""
    w = inputs.config(4)
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w)
    s.init_equilibrium_host(torch.from_numpy(rho).pin_memory(), None)
    k = 3
    s.step(k)
    centers = [(0, 0, 0), (511, 511, 511), (17, 300, 1), (200, 5, 510), (256, 256, 256), (511, 0, 2)]
    err = _subbox_check(lbm, w, s, k, centers)
    print(f"\ntest_config4_channel512_sampled: max|df| vs oracle on the sampled sub-boxes = {err:.2e}")
    assert err <= TOL
    steps = 200
    s.step(steps - k)
    _, uf, d = s.moments()
    prof = uf[0].view(512, 512 * 512).mean(dim=1).cpu().numpy()
    H, F, nu = 512, w.force[0], (w.tau - 0.5) / 3
    z = np.arange(H) + 0.5
    u_an = F * z * (H - z) / (2 * nu)
    for n_ in range(1, 4000, 2):
        u_an -= 4 * F * H * H / (nu * np.pi**3 * n_**3) * np.sin(n_ * np.pi * z / H) * np.exp(-n_ * n_ * np.pi**2 * nu * steps / H**2)
    assert np.linalg.norm(prof - u_an) / np.linalg.norm(u_an) < 1e-2
    assert abs(d[0] / w.N - 1) < 1e-5 and d[7] == 0
    s.close()


@pytest.mark.parametrize("Q", [19, 27])
def test_channel_steady_state_small_H(lbm, Q):
    """configs[4] physics on the converged nz = 16 analogue through the GPU: parabola + BGK slip constant."""
    H, tau, F = 16, 0.9, 1e-7
    nu = (tau - 0.5) / 3
    fk = [P, P, P, P, B, B]
    o, s = make_pair(lbm, (4, 4, H), Q, tau, face_kind=fk, force=(F, 0, 0))
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    o.step(20000)
    s.step(20000)
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
    _, u, _ = s.moments()
    prof = u[0].cpu().numpy().reshape(H, 16).mean(axis=1)
    z = np.arange(H) + 0.5
    ref = F * z * (H - z) / (2 * nu) + F / (2 * nu) * (4 * (tau - 0.5) ** 2 / 3 - 0.25)
    assert np.abs(prof - ref).max() / ref.max() < 1e-9
    s.close()


# --------------------------------------------------------------------------- D2Q9 (S:§8f NEXT-4; Eq. 3-4)

@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_d2q9_taylor_green_decay(lbm, scheme):
    """The paper's printed D2Q9 lattice on a single plane (nz = 1): 2-D Taylor-Green vortex, an exact
    Navier-Stokes solution decaying as exp(-2 nu |k|^2 t), |k|^2 = 2 (2 pi / n)^2; parity with the oracle
    over the whole run and the decay rate from the GPU's own energy history."""
    n, tau, u0, steps = 64, 0.8, 0.02, 300
    rho, u = inputs.taylor_green_2d(n, n, 1, u0)
    o = Oracle(n, n, 1, 9, tau)
    s = lbm.Solver(n, n, 1, 9, tau, scheme=dict(schemes(lbm))[scheme])
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    E = [s.diagnostics()[4]]
    for _ in range(steps // 10):
        s.step(10)
        E.append(s.diagnostics()[4])
    o.step(steps)
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
    nu, k2 = (tau - 0.5) / 3, 2 * (2 * np.pi / n) ** 2
    slope = np.polyfit(10 * np.arange(len(E)), np.log(E), 1)[0]
    assert abs(slope / (-2 * nu * k2) - 1) < 2e-3
    s.close()


def test_d2q9_planes_are_independent(lbm):
    """LBM_D2Q9 with nz > 1: every z-plane is an independent 2-D domain (include/lbm.h)."""
    nx, ny, nz = 40, 24, 3
    f0 = random_f(9, nx * ny * nz, seed=3)
    fk = [B, B, P, P, P, P]
    o, s = make_pair(lbm, (nx, ny, nz), 9, 0.7, face_kind=fk, force=(1e-4, 2e-4, 0))
    o.set_f(f0)
    s.set_populations(dev(f0))
    o.step(6)
    s.step(6)
    got = s.get_populations().cpu().numpy()
    assert np.abs(got - o.get_f()).max() <= TOL
    one = lbm.Solver(nx, ny, 1, 9, 0.7, face_kind=fk, force=(1e-4, 2e-4, 0))
    one.set_populations(dev(f0.reshape(9, nz, ny * nx)[:, 1].copy()))
    one.step(6)
    assert (one.get_populations().cpu().numpy() == got.reshape(9, nz, ny * nx)[:, 1]).all()
    one.close()
    s.close()


# --------------------------------------------------------------------------- fp32-storage variant (S:§8f NEXT-1)

@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_fp32_storage_variant(lbm, scheme):
    """BASELINE.json north_star: populations match the oracle within 2e-5 relative with fp32 storage."""
    w = inputs.config(0)
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau)
    s = lbm.Solver.from_workload(w, scheme=dict(schemes(lbm))[scheme], store=lbm.LBM_STORE_F32)
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    o.step(w.steps)
    s.step(w.steps)
    ref = o.get_f()
    got = s.get_populations().cpu().numpy()
    assert (np.abs(got - ref) / np.abs(ref)).max() <= 2e-5
    s.close()


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_storage_layouts_give_identical_results(lbm, scheme):
    """LBM_LAYOUT_SOA (f[a][z][y][x]) and the default row-interleaved f[z][y][a][x] are two placements of the same
    values: every cell does the same arithmetic, so the canonical populations agree bit for bit — periodic, with
    walls + lid, and with a solid mask under the nodal model."""
    dims = (70, 9, 6)
    N = dims[0] * dims[1] * dims[2]
    rng = np.random.default_rng(5)
    f0 = torch.from_numpy(np.full((19, 1), 1.0 / 19) * (1.0 + 0.1 * rng.uniform(-1, 1, (19, N)))).cuda().reshape(-1)
    geo = torch.from_numpy((rng.uniform(size=N) < 0.05).astype(np.uint8)).cuda()
    cases = [dict(), dict(face_kind=[1, 1, 1, 1, 1, 2], face_u=[[0, 0, 0]] * 5 + [[0.1, 0, 0]]), dict(geo=True, force=(1e-5, 0, 0))]
    for case in cases:
        use_geo = case.pop("geo", False)
        out = []
        for layout in (lbm.LBM_LAYOUT_ROWS, lbm.LBM_LAYOUT_SOA):
            s = lbm.Solver(*dims, 19, 0.7, scheme={"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme], layout=layout, **case)
            if use_geo:
                s.set_geometry(geo, lbm.LBM_WALL_NODAL)
            s.set_populations(f0)
            s.step(5)
            out.append((s.get_populations().clone(), s.moments()[0].clone()))
            s.close()
        assert torch.equal(out[0][0], out[1][0]) and torch.equal(out[0][1], out[1][1])


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_large_box_equals_its_periodic_tile(lbm, scheme):
    """Maximum sizes: 640^3 D3Q19 (Q*N = 4.98e9 stored elements: offsets beyond 2^32, 40 GB per buffer) started from a
    128^3 field tiled 5 x 5 x 5.  A periodic flow whose period divides the box evolves exactly like the small periodic
    box (same arithmetic per cell), so after an odd number of steps rho and u of the large box are the small box's,
    tile by tile, bit for bit — and the small box is compared with the oracle elsewhere in this file."""
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        pytest.skip("needs 120 GB of free device memory")
    n, k, steps = 128, 5, 7
    w = inputs.config(1).scaled(n, steps=steps)
    rho, u = w.fields()
    rho_s = torch.from_numpy(rho).cuda()
    u_s = torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda()
    sch = {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme]
    s = lbm.Solver.from_workload(w, scheme=sch)
    s.init_equilibrium(rho_s, u_s)
    s.step(steps)
    r_small, u_small, d_small = s.moments()
    r_small, u_small = r_small.clone().view(n, n, n), u_small.clone().view(3, n, n, n)
    s.close()
    N = n * k
    big = lbm.Solver(N, N, N, 19, w.tau, scheme=sch)
    rho_b = rho_s.view(n, n, n).repeat(k, k, k).reshape(-1)
    u_b = u_s.view(3, n, n, n).repeat(1, k, k, k).reshape(-1)
    big.init_equilibrium(rho_b, u_b)
    del rho_b, u_b
    big.step(steps)
    r_big, u_big, d_big = big.moments()
    big.close()
    r_big, u_big = r_big.view(N, N, N), u_big.view(3, N, N, N)
    for tz, ty, tx in ((0, 0, 0), (k - 1, k - 1, k - 1), (2, 4, 1), (4, 0, 3)):
        sl = (slice(tz * n, (tz + 1) * n), slice(ty * n, (ty + 1) * n), slice(tx * n, (tx + 1) * n))
        assert torch.equal(r_big[sl], r_small)
        assert torch.equal(u_big[(slice(None),) + sl], u_small)
    assert d_big[7] == 0 and d_big[5] == d_small[5] and d_big[6] == d_small[6]
    assert abs(d_big[0] - k**3 * d_small[0]) <= 1e-12 * d_big[0]


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_large_plane_beyond_32bit_row_offsets_equals_its_tile(lbm, scheme):
    """D2Q9 16384 x 16384 x 1: Q*nx*ny = 2.4e9 >= 2^31, so the row-interleaved layout's 32-bit in-plane offsets x + y*(Q*nx)
    would overflow; lbm_create stores such a grid as a plain structure of arrays instead (include/lbm.h LBM_LAYOUT_ROWS).
    Started from a 2048^2 Taylor-Green field tiled 8 x 8 it must reproduce the small box tile by tile, bit for bit, and
    leave the guard zones around its buffers intact."""
    free, _ = torch.cuda.mem_get_info()
    if free < 80e9:
        pytest.skip("needs 80 GB of free device memory")
    n, k, steps = 2048, 8, 5
    rho, u = inputs.taylor_green_2d(n, n, 1, 0.03)
    rho_s, u_s = dev(rho), dev(u.reshape(-1))
    sch = dict(schemes(lbm))[scheme]
    s = lbm.Solver(n, n, 1, 9, 0.7, scheme=sch)
    s.init_equilibrium(rho_s, u_s)
    s.step(steps)
    r_small, u_small, d_small = s.moments()
    r_small, u_small = r_small.clone().view(n, n), u_small.clone().view(3, n, n)
    s.close()
    N = n * k
    big = lbm.Solver(N, N, 1, 9, 0.7, scheme=sch)
    big.debug_arm(poison=True)
    big.init_equilibrium(rho_s.view(n, n).repeat(k, k).reshape(-1), u_s.view(3, n, n).repeat(1, k, k).reshape(-1))
    big.step(steps)
    r_big, u_big, d_big = big.moments()
    assert big.debug_check() == 0
    big.close()
    assert bool((r_big.view(k, n, k, n) == r_small.view(1, n, 1, n)).all())
    assert bool((u_big.view(3, k, n, k, n) == u_small.view(3, 1, n, 1, n)).all())
    assert d_big[7] == 0 and d_big[5] == d_small[5] and d_big[6] == d_small[6]


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_persistent_kernel_equals_one_launch_per_step(lbm, scheme):
    """lbm_step(n) on a small grid runs in ONE cooperative launch of the persistent kernel (all n steps, a grid-wide
    barrier between them); with lbm_set_persistent(0) it is n launches.  Same cell code: identical bits — periodic,
    cavity with lid, inlet / outlet with a solid mask under the nodal model, odd and even step counts."""
    sch = {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme]
    dims = (48, 20, 12)
    N = dims[0] * dims[1] * dims[2]
    rng = np.random.default_rng(9)
    f0 = torch.from_numpy(np.full((19, 1), 1.0 / 19) * (1.0 + 0.1 * rng.uniform(-1, 1, (19, N)))).cuda().reshape(-1)
    geo = torch.from_numpy((rng.uniform(size=N) < 0.03).astype(np.uint8)).cuda()
    lid = dict(face_kind=[1, 1, 1, 1, 1, 2], face_u=[[0, 0, 0]] * 5 + [[0.1, 0, 0]])
    openx = dict(face_kind=[2, 3, 1, 1, 0, 0], face_u=[[0.03, 0, 0]] + [[0, 0, 0]] * 5, force=(1e-5, 0, 0))
    for case, use_geo in ((dict(), False), (lid, False), (openx, True)):
        out = []
        for on in (1, 0):
            s = lbm.Solver(*dims, 19, 0.7, scheme=sch, **case)
            s.set_persistent(on)
            s.set_two_step(0)  # (without the persistent kernel: one launch per step, not stream_collide_ab2's one per two)
            if use_geo:
                s.set_geometry(geo, lbm.LBM_WALL_NODAL)
            s.set_populations(f0)
            l0 = s.launches
            s.step(7)
            s.step(10)
            out.append((s.get_populations().clone(), s.launches - l0))
            s.close()
        assert torch.equal(out[0][0], out[1][0])
        assert out[1][1] - out[0][1] == 15, out  # 17 step launches became 2


def _two_step_case(lbm, Q, dims, faces, eq, forced, pairs=True):
    nx, ny, nz = dims
    N = nx * ny * nz
    kinds, uspec = FACE_CASES_TWO_STEP[faces]
    fu = face_u_of(uspec)
    force = (1e-5, -2e-6, 3e-6) if forced else None
    f0 = random_f(Q, N, seed=nx + ny + nz + Q)
    o, _s = make_pair(lbm, dims, Q, 0.57, eq=eq, face_kind=kinds, face_u=fu, force=force)
    _s.close()
    o.set_f(f0)
    o.step(7)
    ref = o.get_f()
    o.close()
    out = []
    for on in (2, 0):  # 2: the two-step kernel on any grid it exists for (the default, 1, leaves small grids to the one-step kernel)
        s = lbm.Solver(nx, ny, nz, Q, 0.57, eq=eq_flag(lbm, eq), scheme=lbm.LBM_SCHEME_AB, face_kind=kinds, face_u=fu, force=force)
        s.set_persistent(0)  # (these grids would otherwise run in the persistent kernel)
        s.set_two_step(on)
        s.debug_arm(poison=True)
        s.set_populations(dev(f0).reshape(-1))
        l0 = s.launches
        s.step(4)  # two passes
        s.step(3)  # one pass + one single step
        launches = s.launches - l0
        out.append((s.get_populations().clone(), launches))
        assert s.debug_check() == 0
        s.close()
    assert out[0][1] == (4 if pairs else 7) and out[1][1] == 7, (out[0][1], out[1][1])
    assert torch.equal(out[0][0], out[1][0])
    assert float(np.abs(out[0][0].cpu().numpy().reshape(Q, N) - ref).max()) <= TOL


@pytest.mark.parametrize("dims", [(32, 8, 4), (64, 16, 21), (40, 27, 19), (33, 9, 35), (96, 40, 50), (65, 17, 9), (128, 25, 12)])
@pytest.mark.parametrize("faces", list(FACE_CASES_TWO_STEP))
@pytest.mark.parametrize("eq,forced", [(EQ_STANDARD, False), (EQ_STANDARD, True), (EQ_INCOMP, False), (EQ_INCOMP, True)])
def test_two_step_kernel_equals_single_steps_and_the_oracle(lbm, dims, faces, eq, forced):
    """stream_collide_ab2 (two time steps per pass through HBM: stage 1 on a tile extended by one cell into shared memory,
    stage 2 from there; lbm_set_two_step, default on for fp64 A/B without a solid mask) against the one-step kernel
    — same arithmetic per cell: identical bits — and against the oracle, from random non-equilibrium populations: periodic
    boxes, walls, the lid, moving walls on every face; grids of one tile, of ragged tiles in x and y, more z-chunks than
    one, odd and even step counts.  D3Q19: 32 x 8 tiles, one barrier per plane, register prefetch."""
    _two_step_case(lbm, 19, dims, faces, eq, forced)


@pytest.mark.parametrize("dims", [(16, 8, 4), (48, 16, 21), (40, 27, 19), (17, 9, 35), (96, 40, 50)])
@pytest.mark.parametrize("faces", ["periodic", "channel_z", "couette_z", "inlet_outlet_z"])
@pytest.mark.parametrize("eq,forced", [(EQ_STANDARD, False), (EQ_STANDARD, True), (EQ_INCOMP, False), (EQ_INCOMP, True)])
def test_two_step_kernel_d3q27(lbm, dims, faces, eq, forced):
    """The same for D3Q27: 16 x 8 tiles, two barriers per plane (1 / 2 / 3 slots per e_z class), no prefetch, two blocks
    per SM — periodic boxes, and boxes with z walls (bounce-back, moving) whose x and y faces are periodic: there the
    walls act through ghost planes that stage 1 fills (BJ config 5's boundary set)."""
    _two_step_case(lbm, 27, dims, faces, eq, forced)


@pytest.mark.parametrize("faces", ["cavity", "mixed"])
def test_two_step_mode_leaves_d3q27_with_xy_walls_to_the_one_step_kernel(lbm, faces):
    """D3Q27 with walls in x or y has no two-step kernel (measured: no gain): lbm_step falls back to one launch per step."""
    _two_step_case(lbm, 27, (48, 16, 21), faces, EQ_STANDARD, True, pairs=False)


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("faces", ["periodic", "cavity", "mixed", "couette_z"])
def test_two_step_kernel_on_a_grid_that_fills_the_device(lbm, faces, Q):
    """The same bit-for-bit comparison where every SM runs blocks of stream_collide_ab2 at once and warps of a block drift
    apart between its barriers (320 x 192 x 96 = 5.9 M cells, 1440 blocks in 6 z-chunks, 40 steps): a hazard between
    stage 1 of one plane and stage 2 of the previous one on a shared-memory slot shows up here, not on 10^4 cells."""
    nx, ny, nz = 320, 192, 96
    kinds, uspec = FACE_CASES[faces]
    fu = face_u_of(uspec)
    w = inputs.Workload("fill", nx, ny, nz, Q, 0.55, 40, face_kind=tuple(kinds), face_u=tuple(map(tuple, fu)), u0=0.04, noise=1e-3,
                        force=(1e-6, 0.0, 0.0) if Q == 27 else (0.0, 0.0, 0.0),
                        seed=inputs.SEED_BASE + 77, kind="tgv" if faces == "periodic" else "rest")
    rho, u = w.fields()
    rho_d, u_d = dev(rho), dev(u.reshape(-1))
    out = []
    for on in (1, 0):
        s = lbm.Solver.from_workload(w, scheme=lbm.LBM_SCHEME_AB)
        s.set_two_step(on)
        s.init_equilibrium(rho_d, u_d)
        d0 = s.diagnostics()
        s.step(w.steps)
        out.append((s.get_populations().clone(), s.diagnostics()))
        s.close()
    assert torch.equal(out[0][0], out[1][0])
    assert out[0][1][7] == 0
    if faces != "mixed":
        assert abs(out[0][1][0] - d0[0]) <= 1e-12 * d0[0]  # mass: the lid's +- links cancel (R6)


def test_two_step_default_leaves_small_grids_to_the_one_step_kernel(lbm):
    """lbm_set_two_step's default (1) takes steps in pairs only where the grid gives stream_collide_ab2 at least 1.4 waves of
    blocks (64^3 gives at most 128 blocks of 32 x 8 x 8 cells: one-step kernel; 128^3 gives 576); 2 forces it, 0 switches it
    off."""
    for n, paired in ((64, False), (128, True)):
        s = lbm.Solver(n, n, n, 19, 0.6, scheme=lbm.LBM_SCHEME_AB)
        s.set_persistent(0)
        s.init_equilibrium()
        for mode, expect in ((1, 5 if paired else 10), (2, 5), (0, 10)):
            s.set_two_step(mode)
            l0 = s.launches
            s.step(10)
            assert s.launches - l0 == expect, (n, mode, s.launches - l0)
        s.close()
    with pytest.raises(lbm.LBMError):
        s = lbm.Solver(16, 16, 16, 19, 0.6)
        try:
            s.set_two_step(3)
        finally:
            s.close()


# fp32 storage: the two-cells-per-thread kernel against the one-cell kernel ------------------------------------------
# D2Q9 lives in the x-y plane: its own face mixes (z faces periodic)
FACE_CASES_F32_2D = {
    "periodic": ([P] * 6, None),
    "cavity": ([B, B, B, M, P, P], {3: (0.1, 0.0, 0.0)}),
    "mixed": ([B, M, P, P, P, P], {1: (0.0, 0.03, 0.0)}),
    "inlet_outlet_x": ([M, PR, B, B, P, P], {0: (0.04, 0.0, 0.0)}),
}


@pytest.mark.parametrize("forced", [False, True], ids=["unforced", "forced"])
@pytest.mark.parametrize("faces", ["periodic", "cavity", "mixed", "inlet_outlet_x"])
@pytest.mark.parametrize("Q", [19, 9])
def test_fp32_two_cell_kernel_equals_one_cell_kernel(lbm, Q, faces, forced):
    """stream_collide_ab_f32x2 (the default fp32 A/B kernel of every even-nx D3Q19 / D2Q9 box without a mask: two cells
    per thread) claims the bits of the one-cell kernel.  The one-cell kernel is reached through an all-fluid solid mask
    (the BC_GEO path, which test_returning_to_the_analytic_box shows to be bit-identical to the analytic box in fp64).
    Random non-equilibrium f, so that a wrong wall, wrap or pair link at x = 0 / x = nx-2 cannot hide below a tolerance.
    Row widths: nx = 2*bx exactly (64 with bx = 32; 256 with bx = 128), and nx that is not a multiple of 2*bx (70, 300)."""
    kinds, uspec = (FACE_CASES_TWO_STEP if Q == 19 else FACE_CASES_F32_2D)[faces]
    fu = face_u_of(uspec)
    force = ((1e-5, -2e-6, 3e-6) if Q == 19 else (1e-5, -2e-6, 0.0)) if forced else None
    for dims in ((64, 6, 5), (70, 5, 4), (256, 3, 3), (300, 4, 3)):
        N = dims[0] * dims[1] * dims[2]
        f0 = dev(random_f(Q, N, seed=Q + dims[0]).reshape(-1))
        out = []
        for one_cell in (False, True):
            s = lbm.Solver(*dims, Q, 0.57, scheme=lbm.LBM_SCHEME_AB, store=lbm.LBM_STORE_F32, face_kind=kinds, face_u=fu, force=force)
            if one_cell:
                s.set_geometry(torch.zeros(N, dtype=torch.uint8, device="cuda"), lbm.LBM_WALL_HALFWAY)
            s.set_populations(f0)
            s.step(7)
            out.append(s.get_populations().clone())
            s.close()
        assert bool(torch.isfinite(out[0]).all())
        assert torch.equal(out[0], out[1]), (Q, faces, forced, dims, float((out[0] - out[1]).abs().max()))
