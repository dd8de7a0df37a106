"""GPU parity for the open boundaries (R22; the paper's channel-cylinder example): FACE_PRESSURE
(anti-bounce-back at a prescribed density) and FACE_MOVING with a per-cell wall-velocity profile (velocity inlet),
through the C ABI (lbm_set_face_density, lbm_set_face_velocity) against the CPU oracle, element by element.
Tolerance: max |df| <= 1e-12 (BASELINE.json north_star); fp32 storage <= 2e-5 relative.  `pytest -m gpu` on a B200.
"""
import numpy as np
import pytest

from oracle import Oracle
from oracle.binding import EQ_INCOMP, EQ_STANDARD, WALL_HALFWAY
from paper_2201_11330_b200 import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
TOL = 1e-12
P, B, M, PR = inputs.FACE_PERIODIC, inputs.FACE_BOUNCE, inputs.FACE_MOVING, inputs.FACE_PRESSURE


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


def make_pair(lbm, dims, Q, tau, fk, eq, scheme, store=0, force=None, seed=0, profiles=True, geo=None):
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
    if geo is not None:
        o.set_geometry(geo, WALL_HALFWAY)
        s.set_geometry(torch.from_numpy(np.ascontiguousarray(geo, dtype=np.uint8).reshape(-1)).cuda(), lbm.LBM_WALL_HALFWAY)
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
    with pytest.raises(lbm.LBMError):  # the paper defines no open boundary for its nodal wall model
        s.set_geometry(None, lbm.LBM_WALL_NODAL)
    with pytest.raises(lbm.LBMError):
        s.set_face_density([1.0, float("nan"), 1, 1, 1, 1])
    s.set_face_velocity(0, dev(np.zeros(3 * 64)))
    s.set_face_velocity(0, None)
    s.close()
    with pytest.raises(lbm.LBMError):  # PRESSURE on one face of an axis, periodic on the other
        lbm.Solver(8, 8, 8, 19, 0.8, face_kind=[PR, P, P, P, P, P])


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
