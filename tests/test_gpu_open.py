"""GPU parity for the open boundaries (R22; the paper's channel-cylinder example): FACE_PRESSURE
(anti-bounce-back at a prescribed density) and FACE_MOVING with a per-cell wall-velocity profile (velocity inlet),
through the C ABI (lbm_set_face_density, lbm_set_face_velocity); FACE_SYMMETRY mirror planes (R25; the sphere case's
"symmetric" sides) and open faces next to the nodal wall model (R24) — against the CPU oracle, element by element.
Tolerance: max |df| <= 1e-12 (BASELINE.json north_star); fp32 storage <= 2e-5 relative.  `pytest -m gpu` on a B200.
"""
import numpy as np
import pytest

from oracle import Oracle
from oracle.binding import EQ_INCOMP, EQ_STANDARD, WALL_HALFWAY, WALL_NODAL
from paper_2201_11330_b200 import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
TOL = 1e-12
P, B, M, PR = inputs.FACE_PERIODIC, inputs.FACE_BOUNCE, inputs.FACE_MOVING, inputs.FACE_PRESSURE
S = inputs.FACE_SYMMETRY


@pytest.fixture(scope="module")
def lbm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_11330_b200 import lbm as _lbm
    _lbm.load()
    return _lbm


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def face_cells(face, dims):
    nx, ny, nz = dims
    return [ny * nz, ny * nz, nx * nz, nx * nz, nx * ny, nx * ny][face]


def random_profile(face, dims, seed, amp=0.05):
    rng = np.random.default_rng(seed)
    return amp * rng.uniform(-1, 1, (3, face_cells(face, dims)))


def random_f(Q, N, seed, amp=0.2):
    rng = np.random.default_rng(seed)
    return np.full((Q, 1), 1.0 / Q) * (1.0 + amp * rng.uniform(-1, 1, (Q, N)))


# every face kind next to every other one, corners included (precedence MOVING > BOUNCE > PRESSURE)
MIXES = {
    "inlet_outlet_x": [M, PR, B, B, P, P],
    "pressure_all": [PR] * 6,
    "pressure_z_moving_y": [P, P, M, M, PR, PR],
    "mixed_corners": [M, PR, PR, B, M, PR],
    "outlet_y_lid_z": [B, B, PR, PR, B, M],
}
FACE_RHO = (1.02, 0.97, 1.01, 0.99, 1.03, 0.98)


def make_pair(lbm, dims, Q, tau, fk, eq, scheme, store=0, force=None, seed=0, profiles=True, geo=None, model=WALL_HALFWAY):
    nx, ny, nz = dims
    fu = np.zeros((6, 3))
    for k in range(6):
        if fk[k] == M:
            fu[k] = (0.03 * (k + 1), -0.02, 0.01 * k)
    o = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=fk, face_u=fu, force=force, face_rho=FACE_RHO)
    s = lbm.Solver(nx, ny, nz, Q, tau, eq=lbm.LBM_EQ_INCOMP if eq == EQ_INCOMP else lbm.LBM_EQ_STANDARD,
                   scheme={"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme], store=store,
                   face_kind=fk, face_u=fu, force=force)
    s.set_face_density(FACE_RHO)
    if geo is not None or model != WALL_HALFWAY:
        o.set_geometry(geo, model)
        s.set_geometry(None if geo is None else torch.from_numpy(np.ascontiguousarray(geo, dtype=np.uint8).reshape(-1)).cuda(), model)
    if profiles:
        # every second MOVING face gets a per-cell profile, the others keep the uniform face_u
        for j, k in enumerate([k for k in range(6) if fk[k] == M]):
            if j % 2 == 0:
                prof = random_profile(k, dims, seed + 10 + k)
                o.set_face_velocity(k, prof)
                s.set_face_velocity(k, dev(prof.reshape(-1)))
    return o, s


@pytest.mark.parametrize("scheme", ["ab", "aa"])
@pytest.mark.parametrize("eq", [EQ_STANDARD, EQ_INCOMP])
@pytest.mark.parametrize("Q", [9, 19, 27])
@pytest.mark.parametrize("mix", sorted(MIXES))
def test_open_faces_match_oracle(lbm, mix, Q, eq, scheme):
    """Random non-equilibrium populations, 5 steps (odd: the AA export has to un-swap), ragged box."""
    dims = (37, 11, 1 if Q == 9 else 6)
    fk = list(MIXES[mix])
    if Q == 9:
        fk[4] = fk[5] = P  # one plane: z is periodic
    N = dims[0] * dims[1] * dims[2]
    force = (1e-5, -2e-5, 0.0) if mix == "mixed_corners" else None
    o, s = make_pair(lbm, dims, Q, 0.62, fk, eq, scheme, force=force, seed=3)
    f0 = random_f(Q, N, 7)
    o.set_f(f0)
    s.set_populations(dev(f0))
    for n in (1, 4):
        o.step(n)
        s.step(n)
        err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
        assert err <= TOL, f"{mix} Q{Q} eq{eq} {scheme}: max|df| = {err:.3e} after {s.time} steps"
    rho_o, u_o, d_o = o.moments()
    rho_g, u_g, d_g = s.moments()
    assert np.abs(rho_g.cpu().numpy() - rho_o).max() <= TOL
    assert np.abs(u_g.cpu().numpy() - u_o).max() <= TOL
    assert abs(d_g[0] - d_o[0]) <= 1e-12 * abs(d_o[0])
    s.close()


@pytest.mark.parametrize("mix", ["inlet_outlet_x", "mixed_corners"])
def test_open_faces_fp32_storage(lbm, mix):
    dims = (40, 12, 5)
    o, s = make_pair(lbm, dims, 19, 0.7, MIXES[mix], EQ_STANDARD, "ab", store=lbm.LBM_STORE_F32, seed=5)
    rho = 1.0 + 1e-3 * np.random.default_rng(1).uniform(-1, 1, dims[0] * dims[1] * dims[2])
    o.init_equilibrium(rho, None)
    s.init_equilibrium(dev(rho), None)
    o.step(20)
    s.step(20)
    ref = o.get_f()
    err = np.abs(s.get_populations().cpu().numpy() - ref).max() / np.abs(ref).max()
    assert err <= 2e-5, err
    s.close()


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_open_faces_with_solid_mask(lbm, scheme):
    """The BC_GEO kernels (link mask) with open faces: an obstacle in a channel with inlet and outlet."""
    dims = (48, 20, 1)
    geo = inputs.cylinder_mask(*dims, (12.0, 9.5), 3.0)
    geo.reshape(1, 20, 48)[0, 0:2, 30] = 1  # a stub on the y- wall
    geo.reshape(1, 20, 48)[0, 5, 0] = 1     # a solid node in the inlet plane
    geo.reshape(1, 20, 48)[0, 14, 47] = 1   # and one in the outlet plane
    o, s = make_pair(lbm, dims, 9, 0.56, MIXES["inlet_outlet_x"], EQ_INCOMP, scheme, seed=9, geo=geo)
    rho = inputs.density_noise(*dims, 1e-4, 11)
    o.init_equilibrium(rho, None)
    s.init_equilibrium(dev(rho), None)
    for n in (7, 30):
        o.step(n)
        s.step(n)
        err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
        assert err <= TOL, err
        assert np.abs(s.boundary_force() - o.boundary_force()).max() <= TOL
    s.close()


def test_channel_cylinder_workload_matches_oracle(lbm):
    """inputs.config(7) (the paper's Re = 100 case) shrunk by 2: Solver.from_workload applies the parabolic
    inlet profile, the outlet density and the cylinder; 400 steps against the oracle, drag and lift included."""
    w = inputs.config(7).shrunk(2, steps=400)
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force, face_rho=w.face_rho)
    o.set_geometry(w.geo(), w.wall_model)
    for k, prof in w.face_profiles().items():
        o.set_face_velocity(k, prof)
    o.init_equilibrium(rho, u)
    s = lbm.Solver.from_workload(w)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    o.step(w.steps)
    s.step(w.steps)
    err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
    assert err <= TOL, err
    Fg, Fo = s.boundary_force(), o.boundary_force()
    assert np.abs(Fg - Fo).max() <= TOL
    assert Fo[0] > 0.0  # drag points downstream
    s.close()


def test_open_faces_on_slabs(lbm):
    """z-slabs (D:R21) of a box with open x / y faces and a PRESSURE z+ face: per-cell profiles are indexed by the
    GLOBAL plane; result equals the undivided run bit for bit and the oracle to 1e-12."""
    from paper_2201_11330_b200 import slabs
    dims = (20, 9, 12)
    fk = [M, PR, PR, M, B, PR]
    fu = np.zeros((6, 3))
    fu[0] = (0.04, 0.0, 0.01)
    fu[3] = (0.02, 0.0, -0.01)
    w = inputs.Workload("open_slabs", *dims, 19, 0.66, 6, face_kind=tuple(fk), face_u=tuple(map(tuple, fu)),
                        noise=1e-3, seed=5, kind="rest", face_rho=FACE_RHO)
    profs = {0: random_profile(0, dims, 21), 3: random_profile(3, dims, 22)}
    rho, u = w.fields()
    o = Oracle(*dims, 19, w.tau, face_kind=fk, face_u=fu, face_rho=FACE_RHO)
    for k, pr in profs.items():
        o.set_face_velocity(k, pr)
    o.init_equilibrium(rho, u)
    o.step(w.steps)
    ref = o.get_f()
    whole = lbm.Solver.from_workload(w)
    for k, pr in profs.items():
        whole.set_face_velocity(k, dev(pr.reshape(-1)))
    whole.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    whole.step(w.steps)
    f_whole = whole.get_populations().cpu().numpy()
    whole.close()
    assert np.abs(f_whole - ref).max() <= TOL
    for nslabs in (2, 3):
        g = slabs.SlabGroup(w, nslabs)
        for sl in g.slabs:
            lbm.lbm_set_face_density(sl.h, FACE_RHO)
            for k, pr in profs.items():
                lbm.lbm_set_face_velocity(sl.h, k, dev(pr.reshape(-1)))
        g.init_equilibrium()
        g.step(w.steps)
        f = g.get_populations().cpu().numpy()
        assert np.array_equal(f, f_whole), nslabs
        g.close()


def test_open_face_argument_checks(lbm):
    s = lbm.Solver(8, 8, 8, 19, 0.8, face_kind=[M, PR, B, B, P, P])
    with pytest.raises(lbm.LBMError):  # not a MOVING face
        s.set_face_velocity(1, dev(np.zeros(3 * 64)))
    with pytest.raises(lbm.LBMError):
        s.set_face_velocity(6, None)
    with pytest.raises(lbm.LBMError):
        s.set_face_density([1.0, float("nan"), 1, 1, 1, 1])
    s.set_face_velocity(0, dev(np.zeros(3 * 64)))
    s.set_face_velocity(0, None)
    s.close()
    with pytest.raises(lbm.LBMError):  # PRESSURE on one face of an axis, periodic on the other
        lbm.Solver(8, 8, 8, 19, 0.8, face_kind=[PR, P, P, P, P, P])
    with pytest.raises(lbm.LBMError):  # mirror planes need the A/B scheme
        lbm.Solver(8, 8, 8, 19, 0.8, face_kind=[S, S, P, P, P, P], scheme=lbm.LBM_SCHEME_AA)


# --------------------------------------------------------------------------- the paper's printed drag coefficients
def _paper_drag(golden_dir):
    import os
    rows = {}
    with open(os.path.join(golden_dir, "paper_drag.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, nx, ny, D, cx, om, Re, cd = line.split()
                rows[k] = dict(nx=int(nx), ny=int(ny), D=float(D), cx=float(cx), omega=float(om), Re=float(Re), cd=float(cd))
    return rows


@pytest.mark.parametrize("case,cfg,steps,every", [("case1", 6, 200000, 500), ("case2", 7, 200000, 100)])
def test_channel_cylinder_drag_matches_the_paper(lbm, golden_dir, case, cfg, steps, every):
    """The paper's section-4 example at full size through the CUDA path: C_D = F_x / (rho U^2 r) (Eq. 12) from the
    momentum-exchange force (Eq. 13).  Paper: 2.06 at Re = 20 (steady), "oscillates around 1.46" at Re = 100 (vortex
    street).  Our inlet / outlet / wall formulae are R22's, not the paper's (it prints none), and the cylinder is a
    halfway staircase, so the bar is 5 % — measured: 2.03 and 1.42.  The workload parameters are checked against the
    golden file, the force itself against the oracle in test_channel_cylinder_workload_matches_oracle."""
    ref = _paper_drag(golden_dir)[case]
    w = inputs.config(cfg)
    assert (w.nx, w.ny) == (ref["nx"], ref["ny"]) and w.cylinder[0] == ref["cx"] and 2 * w.cylinder[2] == ref["D"]
    assert abs(1.0 / w.tau - ref["omega"]) < 1e-12
    nu = (w.tau - 0.5) / 3.0
    assert abs(w.inlet_umax * ref["D"] / nu - ref["Re"]) < 1e-9
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    r, U = w.cylinder[2], w.inlet_umax
    hist = []
    for _ in range(steps // every):
        s.step(every)
        hist.append(s.boundary_force() / (U * U * r))
    s.close()
    h = np.array(hist[len(hist) * 3 // 4:])  # last quarter: steady / fully developed shedding
    cd = h[:, 0].mean()
    assert abs(cd - ref["cd"]) <= 0.05 * ref["cd"], (cd, ref["cd"])
    if case == "case1":
        assert np.abs(h[:, 1]).max() < 1e-3            # steady and symmetric: no lift (Re = 20 < 47)
        assert h[:, 0].std() < 0.02 * cd
    else:
        assert h[:, 1].max() > 0.1 and h[:, 1].min() < -0.1   # von Karman street: the lift oscillates (Re > 47)


# --------------------------------------------------------------------------- symmetry planes (R25), nodal + open (R24)
SYM_MIXES = {
    "sphere_case_faces": [M, PR, S, S, P, P],   # inlet, outlet, symmetric sides, periodic top / bottom
    "duct_sym_walls": [M, PR, S, B, B, S],
    "all_kinds": [S, PR, M, B, PR, S],
    "sym_everywhere": [S] * 6,
    "inlet_outlet_walls": [M, PR, B, B, P, P],  # the channel-cylinder faces: R24 under the nodal model
}


def lumps(dims):
    """Solid lumps: one in the interior, one cut by the y- plane, one in the (0,0,0) corner, single nodes."""
    nx, ny, nz = dims
    g = np.zeros((nz, ny, nx), dtype=np.uint8)
    g[nz // 2:nz // 2 + 2, ny // 2 - 1:ny // 2 + 2, nx // 3:nx // 3 + 3] = 1
    g[:, 0:2, nx // 2:nx // 2 + 2] = 1
    g[0, 0, 0] = 1
    g[nz - 1, ny - 1, nx - 2:] = 1
    g[nz - 1, ny // 2, 0] = 1
    return g.reshape(-1)


@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("model", [WALL_HALFWAY, WALL_NODAL], ids=["halfway", "nodal"])
@pytest.mark.parametrize("Q,eq", [(9, EQ_INCOMP), (19, EQ_STANDARD), (27, EQ_INCOMP)])
@pytest.mark.parametrize("mix", sorted(SYM_MIXES))
def test_symmetry_and_nodal_open_faces_match_oracle(lbm, mix, Q, eq, model, store):
    dims = (37, 11, 1 if Q == 9 else 6)
    fk = list(SYM_MIXES[mix])
    if Q == 9:
        fk[4] = fk[5] = P
    N = dims[0] * dims[1] * dims[2]
    force = (1e-5, -2e-5, 0.0) if mix == "all_kinds" else None
    o, s = make_pair(lbm, dims, Q, 0.62, fk, eq, "ab", store=lbm.LBM_STORE_F32 if store == "f32" else 0, force=force,
                     seed=4, geo=lumps(dims), model=model)
    if store == "f64":
        f0 = random_f(Q, N, 8)
        o.set_f(f0)
        s.set_populations(dev(f0))
        # set_populations makes the nodal state consistent with Eq. 10 on both sides
        assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
        for n in (1, 4):
            o.step(n)
            s.step(n)
            err = float(np.abs(s.get_populations().cpu().numpy() - o.get_f()).max())
            assert err <= TOL, f"{mix} Q{Q} eq{eq} model{model}: max|df| = {err:.3e} after {s.time} steps"
        rho_o, u_o, d_o = o.moments()
        rho_g, u_g, d_g = s.moments()
        assert np.abs(rho_g.cpu().numpy() - rho_o).max() <= TOL
        assert np.abs(u_g.cpu().numpy() - u_o).max() <= TOL
        assert np.abs(s.boundary_force() - o.boundary_force()).max() <= TOL
    else:
        rho = 1.0 + 1e-3 * np.random.default_rng(2).uniform(-1, 1, N)
        o.init_equilibrium(rho, None)
        s.init_equilibrium(dev(rho), None)
        o.step(12)
        s.step(12)
        ref = o.get_f()
        assert np.abs(s.get_populations().cpu().numpy() - ref).max() / np.abs(ref).max() <= 2e-5
    s.close()


def test_uniform_flow_between_mirror_planes_stays_uniform(lbm):
    """Free slip through the CUDA path: u = (U,0,0) between symmetry planes is a steady state (no wall friction)."""
    s = lbm.Solver(64, 33, 5, 19, 0.7, face_kind=[P, P, S, S, S, S])
    u = np.zeros((3, s.N))
    u[0] = 0.05
    s.init_equilibrium(None, dev(u.reshape(-1)))
    f0 = s.get_populations().clone()
    s.step(100)
    assert float((s.get_populations() - f0).abs().max()) <= 1e-15
    s.close()


# --------------------------------------------------------------------------- the sphere case with the paper's boundaries
def _oracle_of(w):
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force, face_rho=w.face_rho)
    if w.has_geometry:
        o.set_geometry(w.geo(), w.wall_model)
    for k, prof in w.face_profiles().items():
        o.set_face_velocity(k, prof)
    return o


def test_sphere_case_open_quarter_size_point_A_history(lbm):
    """inputs.config(8) — inlet, outlet, symmetric sides, periodic top / bottom, nodal sphere — with every length
    divided by 4, 400 steps: the paper's own validation (Fig. 7: velocity and pressure at point A, CPU run against
    GPU run, differences 1e-16..1e-17) repeated as oracle against CUDA path at the scaled point A = (18,18,18)."""
    w = inputs.config(8).shrunk(4, steps=400)
    rho, u = w.fields()
    o = _oracle_of(w)
    s = lbm.Solver.from_workload(w)
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    A = 18 + w.nx * (18 + w.ny * 18)
    worst = 0.0
    for _ in range(20):
        o.step(20)
        s.step(20)
        ro, uo, _ = o.moments()
        rg, ug, _ = s.moments()
        worst = max(worst, abs(float(rg[A]) - ro[A]), float(np.abs(ug[:, A].cpu().numpy() - uo[:, A]).max()))
    assert worst <= 1e-13, worst
    assert np.abs(s.get_populations().cpu().numpy() - o.get_f()).max() <= TOL
    assert np.abs(s.boundary_force() - o.boundary_force()).max() <= TOL
    assert o.boundary_force()[0] > 0
    s.close()


def test_sphere_case_open_full_size_first_steps(lbm):
    """inputs.config(8) at the paper's 512 x 128 x 128: every population after 6 steps, point A = (72,72,72), the force."""
    w = inputs.config(8)
    rho, u = w.fields()
    o = _oracle_of(w)
    s = lbm.Solver.from_workload(w)
    o.init_equilibrium(rho, u)
    s.init_equilibrium(dev(rho), dev(u.reshape(-1)))
    o.step(6)
    s.step(6)
    f = s.get_populations()
    ref = o.get_f()
    err = 0.0
    for a in range(w.Q):  # plane by plane: no second 1.8 GB host copy
        err = max(err, float(np.abs(f[a].cpu().numpy() - ref[a]).max()))
    assert err <= TOL, err
    A = 72 + w.nx * (72 + w.ny * 72)
    ro, uo, _ = o.moments()
    rg, ug, _ = s.moments()
    assert abs(float(rg[A]) - ro[A]) <= 1e-14 and float(np.abs(ug[:, A].cpu().numpy() - uo[:, A]).max()) <= 1e-14
    assert np.abs(s.boundary_force() - o.boundary_force()).max() <= TOL
    s.close()
