"""GPU parity for the geometry rows: the solid mask `geo`, the
paper's modified nodal bounce-back (Eq. 10) and the momentum-exchange force (Eq. 13),
through the C ABI (lbm_set_geometry, lbm_boundary_force) against the CPU oracle, element by element.
Tolerance: max |df| <= 1e-12 (BASELINE.json north_star).  Run with `pytest -m gpu` on a B200.
"""
import numpy as np
import pytest

from oracle import Oracle
from oracle.binding import EQ_INCOMP, EQ_STANDARD, WALL_HALFWAY, WALL_NODAL
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
    _lbm.load()
    return _lbm


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def scheme_of(lbm, name):
    return {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[name]


def make_pair(lbm, dims, Q, tau, geo, model, eq=EQ_STANDARD, scheme="ab", face_kind=None, face_u=None, force=None, store=0):
    nx, ny, nz = dims
    o = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=face_kind, face_u=face_u, force=force)
    o.set_geometry(geo, model)
    s = lbm.Solver(nx, ny, nz, Q, tau, eq=lbm.LBM_EQ_INCOMP if eq == EQ_INCOMP else lbm.LBM_EQ_STANDARD,
                   scheme=scheme_of(lbm, scheme), store=store, face_kind=face_kind, face_u=face_u, force=force)
    s.set_geometry(None if geo is None else torch.from_numpy(np.ascontiguousarray(geo, dtype=np.uint8).reshape(-1)).cuda(), model)
    return o, s


def obstacle_mask(dims, seed=0):
    """A sphere, a thick block (has an inactive core under NODAL), a plate touching a face, single solid nodes
    and a single fluid pocket inside the block."""
    nx, ny, nz = dims
    g = inputs.sphere_mask(nx, ny, nz, (0.3 * nx, 0.55 * ny, 0.5 * nz), 0.22 * min(dims)).reshape(nz, ny, nx).copy()
    g[nz // 2:nz // 2 + 5, 1:7, nx - 9:nx - 2] = 1
    g[nz // 2 + 2, 3, nx - 6] = 0      # a one-node fluid pocket
    g[0:2, :, nx // 2] = 1             # a plate on the z- face
    rng = np.random.default_rng(seed)
    for _ in range(6):
        g[rng.integers(nz), rng.integers(ny), rng.integers(nx)] = 1
    g[0, 0, 0] = 1
    g[nz - 1, ny - 1, nx - 1] = 1
    return g.reshape(-1)


def random_f(Q, N, seed, amp=0.2):
    rng = np.random.default_rng(seed)
    return np.full((Q, 1), 1.0 / Q) * (1.0 + amp * rng.uniform(-1, 1, (Q, N)))


FACES = {
    "periodic": ([P] * 6, None),
    "duct": ([P, P, B, B, B, B], None),
    "cavity": ([B, B, B, B, B, M], {5: (0.1, 0.0, 0.0)}),
}


def face_u_of(spec):
    fu = np.zeros((6, 3))
    for k, v in (spec or {}).items():
        fu[k] = v
    return fu


# --------------------------------------------------------------------------- element-wise parity with a mask

@pytest.mark.parametrize("scheme", ["ab", "aa"])
@pytest.mark.parametrize("model", [WALL_HALFWAY, WALL_NODAL], ids=["halfway", "nodal"])
@pytest.mark.parametrize("faces", list(FACES))
@pytest.mark.parametrize("Q,eq,forced", [(19, EQ_STANDARD, False), (19, EQ_INCOMP, True), (27, EQ_STANDARD, True),
                                         (27, EQ_INCOMP, False), (9, EQ_STANDARD, True)])
def test_random_populations_with_mask(lbm, scheme, model, faces, Q, eq, forced):
    """Ragged 37x21x13 grid with obstacles, random non-equilibrium populations, compared after 1, 3 and 7 steps
    (odd counts: the AA scheme is compared in its swapped phase), then moments, diagnostics and Eq. 13."""
    dims = (37, 21, 13)
    N = dims[0] * dims[1] * dims[2]
    fk, fu = FACES[faces]
    geo = obstacle_mask(dims, seed=Q)
    F = (2e-4, -1e-4, 3e-4 if Q != 9 else 0.0) if forced else None
    o, s = make_pair(lbm, dims, Q, 0.77, geo, model, eq, scheme, fk, face_u_of(fu), F)
    f0 = random_f(Q, N, seed=Q + 7 * eq)
    o.set_f(f0)
    s.set_populations(dev(f0))
    # canonical state right after the import: Eq. 10 already holds on wall nodes (D:R17), inactive nodes report 0
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() == 0.0
    for nsteps in (1, 2, 4):
        o.step(nsteps)
        s.step(nsteps)
        assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
        Fo = o.boundary_force()
        Fg = s.boundary_force()
        np.testing.assert_allclose(Fg, Fo, rtol=0, atol=1e-12 * max(1.0, np.abs(Fo).max()))
        assert np.abs(Fo).max() > 1e-3  # the obstacles really carry a load in this noisy state
    rho, u, d = s.moments()
    ro, uo, do = o.moments()
    act = o.active().astype(bool)
    assert (rho.cpu().numpy()[~act] == 0).all() and (u.cpu().numpy()[:, ~act] == 0).all()
    assert np.abs(rho.cpu().numpy() - ro).max() <= 1e-13
    assert np.abs(u.cpu().numpy() - uo).max() <= 1e-13
    np.testing.assert_allclose(d[:5], do[:5], rtol=1e-12, atol=1e-12)
    np.testing.assert_allclose(d[5:7], do[5:7], rtol=1e-14)
    assert d[7] == do[7] == 0
    s.close()


@pytest.mark.parametrize("scheme", ["ab", "aa"])
@pytest.mark.parametrize("model", [WALL_HALFWAY, WALL_NODAL], ids=["halfway", "nodal"])
def test_fp32_storage_with_mask(lbm, scheme, model):
    dims = (24, 20, 16)
    geo = obstacle_mask(dims)
    o, s = make_pair(lbm, dims, 19, 0.8, geo, model, scheme=scheme, force=(1e-5, 0, 0), store=lbm.LBM_STORE_F32)
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    o.step(51)
    s.step(51)
    ref, got = o.get_f(), s.get_populations().cpu().numpy()
    act = o.active().astype(bool)
    assert (np.abs(got - ref)[:, act] / np.abs(ref[:, act])).max() <= 2e-5
    assert (got[:, ~act] == 0).all()
    np.testing.assert_allclose(s.boundary_force(), o.boundary_force(), rtol=1e-3, atol=1e-8)
    s.close()


@pytest.mark.parametrize("scheme", ["ab", "aa"])
@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_INCOMP)])
def test_nodal_init_equilibrium_is_consistent_with_eq10(lbm, scheme, Q, eq):
    """InitPDF under the nodal model (D:R17): wall nodes already satisfy Eq. 10 at t = 0, on both sides."""
    dims = (20, 9, 11)
    N = dims[0] * dims[1] * dims[2]
    rng = np.random.default_rng(11)
    rho = 1 + 0.05 * rng.standard_normal(N)
    u = 0.05 * rng.standard_normal((3, N))
    geo = obstacle_mask(dims)
    o, s = make_pair(lbm, dims, Q, 0.8, geo, WALL_NODAL, eq, scheme, [P, P, B, B, B, B])
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= 1e-15
    s.close()


def test_nodal_walls_without_a_mask(lbm):
    """geo = NULL with LBM_WALL_NODAL: the first / last planes of the BOUNCE faces are the wall nodes."""
    dims = (6, 5, 17)
    o, s = make_pair(lbm, dims, 19, 0.9, None, WALL_NODAL, face_kind=[P, P, P, P, B, B], force=(1e-6, 0, 0))
    o.init_equilibrium(None, None)
    s.init_equilibrium(None, None)
    o.step(300)
    s.step(300)
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
    s.close()


def test_returning_to_the_analytic_box(lbm):
    """(NULL, HALFWAY) drops the mask: the result equals a solver that never had a geometry, bit for bit; an
    all-fluid mask gives the same populations through the BC_GEO kernels."""
    dims = (33, 10, 9)
    N = dims[0] * dims[1] * dims[2]
    fk = [B, B, P, P, B, B]
    f0 = random_f(19, N, seed=2)
    res = []
    for mode in ("plain", "dropped", "allfluid"):
        s = lbm.Solver(*dims, 19, 0.7, face_kind=fk, force=(1e-4, 0, 0))
        if mode == "dropped":
            s.set_geometry(torch.from_numpy(obstacle_mask(dims)).cuda(), lbm.LBM_WALL_NODAL)
            s.set_geometry(None, lbm.LBM_WALL_HALFWAY)
        if mode == "allfluid":
            s.set_geometry(torch.zeros(N, dtype=torch.uint8).cuda(), lbm.LBM_WALL_HALFWAY)
        s.set_populations(dev(f0))
        s.step(5)
        res.append(s.get_populations().cpu().numpy())
        s.close()
    assert (res[0] == res[1]).all() and (res[0] == res[2]).all()


def test_geometry_argument_errors(lbm):
    s = lbm.Solver(8, 8, 8, 19, 0.8, face_kind=[B, B, B, B, B, M], face_u=face_u_of({5: (0.1, 0, 0)}))
    with pytest.raises(lbm.LBMError) as e:
        s.set_geometry(None, 7)
    assert e.value.code == lbm.LBM_EINVAL
    with pytest.raises(lbm.LBMError):
        s.boundary_force()  # no geometry
    s.set_geometry(torch.zeros(512, dtype=torch.uint8), lbm.LBM_WALL_HALFWAY)  # host pointer path
    s.init_equilibrium()
    with pytest.raises(lbm.LBMError):
        s.boundary_force()  # no step yet
    s.step(1)
    assert (s.boundary_force() == 0).all()  # no solid nodes
    s.close()


def test_host_and_device_masks_agree(lbm):
    dims = (20, 12, 10)
    geo = obstacle_mask(dims)
    res = []
    for host in (False, True):
        s = lbm.Solver(*dims, 27, 0.8, force=(1e-5, 0, 0))
        g = torch.from_numpy(geo)
        s.set_geometry(g if host else g.cuda(), lbm.LBM_WALL_NODAL)
        s.init_equilibrium()
        s.step(9)
        res.append((s.get_populations().cpu().numpy(), s.boundary_force()))
        s.close()
    assert (res[0][0] == res[1][0]).all() and (res[0][1] == res[1][1]).all()


# --------------------------------------------------------------------------- physics through the GPU alone

@pytest.mark.parametrize("model", [WALL_HALFWAY, WALL_NODAL], ids=["halfway", "nodal"])
def test_momentum_exchange_balances_fluid_momentum_on_gpu(lbm, model):
    """Eq. 13 on the GPU against the exact momentum balance of the fluid region, evaluated from the GPU's own
    moment fields (not from the force kernel): sum_R e f (t+1) - sum_R e f (t) = |R| F - F_wall."""
    n = 40
    Fb = np.array([3e-5, -1e-5, 2e-5])
    geo = inputs.sphere_mask(n, n, n, (18.3, 20.1, 19.6), 7.6)
    fluid = torch.from_numpy(geo == 0).cuda()
    s = lbm.Solver(n, n, n, 19, 0.8, force=Fb)
    s.set_geometry(torch.from_numpy(geo).cuda(), model)
    rng = np.random.default_rng(1)
    s.init_equilibrium(dev(1 + 0.01 * rng.standard_normal(n**3)), dev(0.02 * rng.standard_normal(3 * n**3)))

    def momentum():
        rho, u, _ = s.moments()
        return np.array([float((rho[fluid] * u[c][fluid]).sum()) for c in range(3)])

    s.step(3)
    for _ in range(3):
        m0 = momentum()
        s.step(1)
        m1 = momentum()
        Fw = s.boundary_force()
        np.testing.assert_allclose(float(fluid.sum()) * Fb - (m1 - m0), Fw, rtol=0, atol=1e-10 * np.abs(Fw).max() + 1e-13)
    s.close()


def test_steady_drag_equals_total_body_force_on_gpu(lbm):
    n = 24
    Fb = np.array([1e-5, 0, 0])
    geo = inputs.sphere_mask(n, n, n, (11.5, 11.5, 11.5), 5.2)
    s = lbm.Solver(n, n, n, 19, 1.0, force=Fb)
    s.set_geometry(torch.from_numpy(geo).cuda(), lbm.LBM_WALL_HALFWAY)
    s.init_equilibrium()
    s.step(12000)
    Fw = s.boundary_force()
    assert Fw[0] == pytest.approx(float((geo == 0).sum()) * Fb[0], rel=1e-6)
    assert abs(Fw[1]) < 1e-12 and abs(Fw[2]) < 1e-12
    s.close()


# --------------------------------------------------------------------------- the paper's sphere case

def _oracle_of(w):
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force)
    if w.has_geometry:
        o.set_geometry(w.geo(), w.wall_model)
    return o


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_sphere_case_quarter_size_long_run(lbm, scheme):
    """inputs.config(5) with every length divided by 4 (128 x 32 x 32, sphere radius 2), 400 steps."""
    w = inputs.config(5).shrunk(4, steps=400)
    rho, u = w.fields()
    o = _oracle_of(w)
    s = lbm.Solver.from_workload(w, scheme=scheme_of(lbm, scheme))
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    o.step(w.steps)
    s.step(w.steps)
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
    np.testing.assert_allclose(s.boundary_force(), o.boundary_force(), rtol=1e-10, atol=1e-13)  # sum of O(0.1) terms that cancel
    s.close()


def test_sphere_case_full_size_first_steps(lbm):
    """inputs.config(5) at the paper's full 512 x 128 x 128 size (D3Q27, Eq. 5, nodal sphere of radius 8): every
    population after 6 steps, the probe point A = (72,72,72) of P:470, and the momentum-exchange force."""
    w = inputs.config(5)
    rho, u = w.fields()
    o = _oracle_of(w)
    s = lbm.Solver.from_workload(w)
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    o.step(6)
    s.step(6)
    got = s.get_populations().cpu().numpy()
    ref = o.get_f()
    assert np.abs(got - ref).max() <= TOL
    A = 72 + w.nx * (72 + w.ny * 72)
    rg, ug, _ = s.moments()
    ro, uo, _ = o.moments()
    # P:470 reports CPU-vs-GPU differences of 1e-16..1e-17 at this point; sums of 27 O(0.1) populations in another order
    assert abs(float(rg[A]) - ro[A]) <= 1e-15 and np.abs(ug[:, A].cpu().numpy() - uo[:, A]).max() <= 1e-15
    np.testing.assert_allclose(s.boundary_force(), o.boundary_force(), rtol=1e-10, atol=1e-12)  # ~2000 O(0.1) terms that cancel
    s.close()
