"""Pins for the CPU oracle (no GPU needed): every part of oracle/lbm_oracle.cpp is checked
against something other than itself — values the paper prints (tests/golden, cited there),
closed forms, invariants, and an independent brute-force gather on tiny grids.

P:n = /root/reference/PAPER.md line n (quoted in the golden files; the reference is never
read at run time).  D:Rk = DESIGN.md reading k.
"""
import itertools
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import Oracle, feq, lattice
from oracle.binding import EQ_INCOMP, EQ_STANDARD, FACE_BOUNCE, FACE_MOVING, FACE_PERIODIC
from paper_2201_11330_b200 import inputs

# --------------------------------------------------------------------------- golden


def _read_golden_d2q9(golden_dir):
    rows = {}
    with open(os.path.join(golden_dir, "d2q9_eq3_eq4.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            key, *vals = line.split()
            rows[key] = vals
    ex = [int(v) for v in rows["ex"]]
    ey = [int(v) for v in rows["ey"]]
    t = [float(Fraction(v)) for v in rows["t"]]
    return ex, ey, t


def _read_constants(golden_dir):
    out = {}
    with open(os.path.join(golden_dir, "paper_constants.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            out[k] = float(v)
    return out


def test_d2q9_equals_paper_eq3_eq4(golden_dir):
    """the oracle's generator with Q=9 must print the paper's own table."""
    ex, ey, t = _read_golden_d2q9(golden_dir)
    e, w = lattice(9)
    assert e[:, 0].tolist() == ex
    assert e[:, 1].tolist() == ey
    assert e[:, 2].tolist() == [0] * 9
    np.testing.assert_allclose(w, t, rtol=0, atol=1e-17)


@pytest.mark.parametrize("Q", [19, 27])
def test_3d_sets_restrict_to_paper_d2q9_order(Q, golden_dir):
    """D:R4: the 3-D numbering extends Eq. 3's rule — its e_z = 0 sub-list is Eq. 3 in order;
    for D3Q27 the renormalised weights of that sub-list are Eq. 4."""
    ex, ey, t = _read_golden_d2q9(golden_dir)
    e, w = lattice(Q)
    sel = e[:, 2] == 0
    assert e[sel, 0].tolist() == ex and e[sel, 1].tolist() == ey
    if Q == 27:
        np.testing.assert_allclose(w[sel] / w[sel].sum(), t, rtol=1e-15)


@pytest.mark.parametrize("Q", [9, 19, 27])
def test_opposite_is_m_minus_1_minus_alpha(Q):
    """alpha-bar = m - 1 - alpha; the rest particle sits in the middle."""
    e, w = lattice(Q)
    for a in range(Q):
        assert (e[Q - 1 - a] == -e[a]).all()
        assert w[Q - 1 - a] == w[a]
    assert (e[(Q - 1) // 2] == 0).all()
    assert len({tuple(v) for v in e.tolist()}) == Q
    assert Q != 19 or (np.abs(e).sum(axis=1) <= 2).all()


@pytest.mark.parametrize("Q", [19, 27])
def test_lattice_isotropy(Q):
    """Moment identities that fix the weights (c_s^2 = 1/3): orders 0..5."""
    e, w = lattice(Q)
    e = e.astype(float)
    d = np.eye(3)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs(np.einsum("q,qi->i", w, e)).max() < 1e-16
    np.testing.assert_allclose(np.einsum("q,qi,qj->ij", w, e, e), d / 3, atol=1e-16)
    assert np.abs(np.einsum("q,qi,qj,qk->ijk", w, e, e, e)).max() < 1e-16
    iso4 = (np.einsum("ij,kl->ijkl", d, d) + np.einsum("ik,jl->ijkl", d, d) + np.einsum("il,jk->ijkl", d, d)) / 9
    np.testing.assert_allclose(np.einsum("q,qi,qj,qk,ql->ijkl", w, e, e, e, e), iso4, atol=1e-16)
    assert np.abs(np.einsum("q,qi,qj,qk,ql,qm->ijklm", w, e, e, e, e, e)).max() < 1e-16


# --------------------------------------------------------------------------- equilibrium


@pytest.mark.parametrize("Q", [19, 27])
def test_equilibrium_moments_eq2(Q):
    """Eq. 2: sum feq = rho, sum e feq = rho u, sum e e feq = rho/3 I + rho u u.
    The second moment pins the printed constants 3, 4.5, 1.5 and any sign or index slip."""
    e, _ = lattice(Q)
    e = e.astype(float)
    rng = np.random.default_rng(1)
    for _ in range(5):
        rho = 1 + 0.1 * rng.standard_normal()
        u = 0.1 * rng.standard_normal(3)
        fe = feq(Q, EQ_STANDARD, rho, u)
        assert abs(fe.sum() - rho) < 1e-15
        np.testing.assert_allclose(fe @ e, rho * u, atol=1e-16)
        np.testing.assert_allclose(np.einsum("q,qi,qj->ij", fe, e, e), rho / 3 * np.eye(3) + rho * np.outer(u, u), atol=1e-16)


@pytest.mark.parametrize("Q", [19, 27])
def test_equilibrium_moments_eq5(Q, golden_dir):
    """Eq. 5: sum feq = p/c_s^2, sum e feq = rho0 u, sum e e feq = p I + rho0 u u, rho0 = 1."""
    rho0 = _read_constants(golden_dir)["rho0"]
    e, _ = lattice(Q)
    e = e.astype(float)
    rng = np.random.default_rng(2)
    for _ in range(5):
        p3 = 1 + 0.1 * rng.standard_normal()  # p / c_s^2
        u = 0.1 * rng.standard_normal(3)
        fe = feq(Q, EQ_INCOMP, p3, u)
        assert abs(fe.sum() - p3) < 1e-15
        np.testing.assert_allclose(fe @ e, rho0 * u, atol=1e-16)
        np.testing.assert_allclose(np.einsum("q,qi,qj->ij", fe, e, e), p3 / 3 * np.eye(3) + rho0 * np.outer(u, u), atol=1e-16)


def test_equilibrium_paper_code_form(golden_dir):
    """P:375-376 prints feq = t*(p*3 + rho0*(3 edu + 4.5 edu^2 - 1.5 udu)); at u = 0 this is t*p*3 and
    Eq. 2 gives t*rho; along a single axis the three printed constants separate."""
    c = _read_constants(golden_dir)
    e, w = lattice(19)
    ux = 0.07
    fe = feq(19, EQ_INCOMP, 1.3, [ux, 0, 0])
    plus = [a for a in range(19) if tuple(e[a]) == (1, 0, 0)][0]
    minus = 18 - plus
    rest = 9
    # antisymmetric part isolates inv_cs2, symmetric part isolates half_inv_cs4 - half_inv_cs2, rest isolates half_inv_cs2
    assert abs((fe[plus] - fe[minus]) / (2 * w[plus]) - c["inv_cs2"] * ux) < 1e-16
    assert abs(fe[rest] / w[rest] - (1.3 - c["half_inv_cs2"] * ux * ux)) < 1e-15
    assert abs((fe[plus] + fe[minus]) / (2 * w[plus]) - (1.3 + (c["half_inv_cs4"] - c["half_inv_cs2"]) * ux * ux)) < 1e-15


@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_STANDARD), (19, EQ_INCOMP), (27, EQ_INCOMP)])
def test_equilibrium_is_fixed_point_of_collision(Q, eq):
    """BASELINE.json north_star: the equilibrium is a fixed point of Eq. 6."""
    n = 6
    rng = np.random.default_rng(3)
    rho = 1 + 0.05 * rng.standard_normal(n**3)
    u = 0.05 * rng.standard_normal((3, n**3))
    o = Oracle(n, n, n, Q, tau=0.6, eq=eq)
    o.init_equilibrium(rho, u)
    f0 = o.get_f()
    o.collision()
    assert np.abs(o.get_fb() - f0).max() < 4e-16


@pytest.mark.parametrize("Q", [19, 27])
def test_eq5_equals_eq2_at_unit_density(Q):
    u = [0.03, -0.02, 0.05]
    np.testing.assert_allclose(feq(Q, EQ_INCOMP, 1.0, u), feq(Q, EQ_STANDARD, 1.0, u), rtol=0, atol=1e-16)


def test_omega_from_tau(golden_dir):
    """D:R1 / P:196: API tau = tau_paper + 1/2, omega = 1/tau.  With the paper's omega = 1.8
    (tau_paper = 1/1.8 - 0.5 = nu/c_s^2, Eq. 11) one collision must relax a non-equilibrium part by 1 - 1.8."""
    om = _read_constants(golden_dir)["omega_case1"]
    o = Oracle(4, 4, 4, 19, tau=1.0 / om)
    f = o.get_f()
    e, w = lattice(19)
    # a perturbation with zero mass and momentum: +d on (1,0,0),(-1,0,0), -2d on rest
    f[:] = w[:, None]
    px = [a for a in range(19) if tuple(e[a]) == (1, 0, 0)][0]
    d = 1e-3
    f[px] += d
    f[18 - px] += d
    f[9] -= 2 * d
    o.set_f(f)
    o.collision()
    fb = o.get_fb()
    np.testing.assert_allclose(fb[px] - w[px], (1 - om) * d, atol=1e-16)
    np.testing.assert_allclose(fb[9] - w[9], (1 - om) * (-2 * d), atol=1e-16)


# --------------------------------------------------------------------------- conservation / forcing


@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_STANDARD), (19, EQ_INCOMP)])
def test_mass_momentum_conserved_periodic(Q, eq):
    """BASELINE.json north_star: mass and momentum conserved to round-off on periodic domains."""
    nx, ny, nz = 12, 10, 8
    rng = np.random.default_rng(4)
    e, w = lattice(Q)
    f = w[:, None] * (1 + 0.1 * rng.standard_normal((Q, nx * ny * nz)))
    o = Oracle(nx, ny, nz, Q, tau=0.7, eq=eq)
    o.set_f(f)
    m0 = f.sum()
    p0 = e.T.astype(float) @ f.sum(axis=1)
    o.step(100)
    f1 = o.get_f()
    assert abs(f1.sum() - m0) / m0 < 1e-13
    np.testing.assert_allclose(e.T.astype(float) @ f1.sum(axis=1), p0, atol=1e-11)
    # the diagnostics agree with the direct sums
    _, _, d = o.moments(False)
    assert abs(d[0] - f1.sum()) / m0 < 1e-14


@pytest.mark.parametrize("Q", [19, 27])
def test_forcing_adds_exactly_F_per_cell_per_step(Q):
    """D:R7: Guo forcing on a periodic box increases sum e f by F*N per step, mass unchanged."""
    n = 8
    F = np.array([1e-5, -2e-5, 3e-5])
    rng = np.random.default_rng(5)
    e, w = lattice(Q)
    o = Oracle(n, n, n, Q, tau=0.9, force=F)
    rho = 1 + 0.01 * rng.standard_normal(n**3)
    u = 0.01 * rng.standard_normal((3, n**3))
    o.init_equilibrium(rho, u)
    f0 = o.get_f()
    steps = 50
    o.step(steps)
    f1 = o.get_f()
    gain = e.T.astype(float) @ (f1.sum(axis=1) - f0.sum(axis=1))
    np.testing.assert_allclose(gain, F * n**3 * steps, rtol=1e-11)
    assert abs(f1.sum() - f0.sum()) / f0.sum() < 1e-14


# --------------------------------------------------------------------------- viscosity


def test_taylor_green_decay_config0():
    """BASELINE.json configs[0]: kinetic energy ~ exp(-2 nu k^2 t), nu = (tau - 1/2)/3, |k|^2 = 3 (2 pi/n)^2
    (D:R11).  Slope of ln E over steps 10..100 within 3 % at 32^3; mass/momentum drift at round-off."""
    w = inputs.config(0)
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau)
    o.init_equilibrium(rho, u)
    d0 = o.moments(False)[2]
    E = [d0[4]]
    for _ in range(w.steps):
        o.step(1)
        E.append(o.moments(False)[2][4])
    d1 = o.moments(False)[2]
    nu = (w.tau - 0.5) / 3
    k2 = 3 * (2 * np.pi / w.nx) ** 2
    slope = np.polyfit(np.arange(10, 101), np.log(E[10:101]), 1)[0]
    assert abs(slope / (-2 * nu * k2) - 1) < 0.03
    assert abs(d1[0] - d0[0]) / d0[0] < 1e-13
    np.testing.assert_allclose(d1[1:4], d0[1:4], atol=1e-11)
    assert d1[7] == 0


@pytest.mark.parametrize("Q", [19, 27])
def test_taylor_green_2d_second_order(Q):
    """Exact 2-D Taylor-Green solution (z-invariant on the 3-D lattice): the error of the measured decay
    rate against nu |k|^2, |k|^2 = 2 (2 pi/n)^2, falls ~4x per doubling of n (second-order method)."""
    tau, u0 = 0.8, 0.01
    nu = (tau - 0.5) / 3
    errs = []
    for n in (16, 32):
        rho, u = inputs.taylor_green_2d(n, n, 2, u0)
        o = Oracle(n, n, 2, Q, tau)
        o.init_equilibrium(rho, u)
        steps = int(round(0.5 / (nu * 2 * (2 * np.pi / n) ** 2)))
        o.step(steps // 4)
        a0 = np.abs(o.moments()[1][0]).max()
        o.step(steps)
        a1 = np.abs(o.moments()[1][0]).max()
        rate = -np.log(a1 / a0) / steps
        errs.append(abs(rate / (nu * 2 * (2 * np.pi / n) ** 2) - 1))
    assert errs[0] < 1e-2 and errs[1] < 2.5e-3
    assert 3.0 < errs[0] / errs[1] < 5.0


# --------------------------------------------------------------------------- walls


def _channel(Q, H, tau, F, steps, eq=EQ_STANDARD):
    fk = [FACE_PERIODIC] * 4 + [FACE_BOUNCE, FACE_BOUNCE]
    o = Oracle(4, 4, H, Q, tau, eq=eq, face_kind=fk, force=[F, 0, 0])
    o.init_equilibrium(None, None)
    o.step(steps)
    _, u, d = o.moments()
    return u[0].reshape(H, 4, 4), d


@pytest.mark.parametrize("Q", [19, 27])
def test_poiseuille_steady_profile(Q):
    """BASELINE.json configs[4] physics on a small-H analogue (D:R9): halfway bounce-back walls + Guo force
    converge to the parabola u(z) = F z (H - z)/(2 nu), z = k + 1/2, plus the known BGK wall-slip constant
    (F/2nu)(4 Lambda/3 - 1/4), Lambda = (tau - 1/2)^2."""
    H, tau, F = 16, 0.9, 1e-7
    nu = (tau - 0.5) / 3
    ux, d = _channel(Q, H, tau, F, 20000)
    z = np.arange(H) + 0.5
    parabola = F * z * (H - z) / (2 * nu)
    slip = F / (2 * nu) * (4 * (tau - 0.5) ** 2 / 3 - 0.25)
    prof = ux.mean(axis=(1, 2))
    assert np.abs(ux - prof[:, None, None]).max() < 1e-18 + 1e-12 * prof.max()  # x,y invariant
    assert np.abs(prof - (parabola + slip)).max() / parabola.max() < 1e-9
    assert np.abs(prof - parabola).max() / parabola.max() < 2e-3  # the bare parabola BASELINE.json names
    assert abs(d[0] - 4 * 4 * H) / (4 * 4 * H) < 1e-12  # walls do not leak mass (round-off drift only, 20000 steps)


def test_poiseuille_startup_series():
    """D:R9: before steady state the plane-averaged profile follows the start-up series
    u(z,t) = F z(H-z)/(2nu) - sum_{n odd} 4 F H^2/(nu pi^3 n^3) sin(n pi z/H) exp(-n^2 pi^2 nu t/H^2)."""
    H, tau, F, steps = 32, 0.9, 1e-7, 600
    nu = (tau - 0.5) / 3
    ux, _ = _channel(19, H, tau, F, steps)
    z = np.arange(H) + 0.5
    u_an = F * z * (H - z) / (2 * nu)
    for n in range(1, 400, 2):
        u_an -= 4 * F * H * H / (nu * np.pi**3 * n**3) * np.sin(n * np.pi * z / H) * np.exp(-n * n * np.pi**2 * nu * steps / H**2)
    prof = ux.mean(axis=(1, 2))
    assert np.linalg.norm(prof - u_an) / np.linalg.norm(u_an) < 5e-3


@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_STANDARD), (19, EQ_INCOMP)])
def test_couette_exact_linear_profile(Q, eq):
    """D:R6 (Ladd moving wall): planar Couette flow between a resting wall (z-) and a wall moving with U
    (z+), both half a cell outside the end nodes, has the exact steady state u_x = U (k + 1/2)/H."""
    H, U = 8, 0.05
    fk = [FACE_PERIODIC] * 4 + [FACE_BOUNCE, FACE_MOVING]
    fu = np.zeros((6, 3))
    fu[5] = [U, 0, 0]
    o = Oracle(4, 4, H, Q, tau=0.8, eq=eq, face_kind=fk, face_u=fu)
    o.init_equilibrium(None, None)
    o.step(4000)
    _, u, d = o.moments()
    prof = u[0].reshape(H, 16).mean(axis=1)
    np.testing.assert_allclose(prof, U * (np.arange(H) + 0.5) / H, atol=1e-13)
    assert np.abs(u[1:]).max() < 1e-14
    assert abs(d[0] - 16 * H) / (16 * H) < 1e-12  # round-off drift only, 4000 steps


def test_cavity_mass_and_mirror_symmetry():
    """BASELINE.json configs[2] on an 8^3 analogue: five resting walls + lid at z+ moving along x.
    Total mass is constant (the +/- lid terms cancel; the lid-takes-precedence tie-break at the lid's
    edges keeps every pair complete) and u_y is antisymmetric under y -> ny-1-y."""
    n = 8
    w = inputs.config(2)
    o = Oracle(n, n, n, 19, w.tau, face_kind=w.face_kind, face_u=w.face_u)
    o.init_equilibrium(None, None)
    o.step(200)
    rho, u, d = o.moments()
    assert abs(d[0] - n**3) / n**3 < 1e-13
    uy = u[1].reshape(n, n, n)
    ux = u[0].reshape(n, n, n)
    assert np.abs(uy + uy[:, ::-1, :]).max() < 1e-15
    assert np.abs(ux - ux[:, ::-1, :]).max() < 1e-15
    assert ux[-1].mean() > 1e-3  # the lid actually drags the fluid along +x


# --------------------------------------------------------------------------- brute force on 4^3

# Hand-written D3Q19 list (not generated): (e_x, e_y, e_z) in the documented order.
_E19 = [(-1, -1, 0), (-1, 0, -1), (-1, 0, 0), (-1, 0, 1), (-1, 1, 0),
        (0, -1, -1), (0, -1, 0), (0, -1, 1), (0, 0, -1), (0, 0, 0), (0, 0, 1), (0, 1, -1), (0, 1, 0), (0, 1, 1),
        (1, -1, 0), (1, 0, -1), (1, 0, 0), (1, 0, 1), (1, 1, 0)]


def _brute_step(f, dims, E, T, omega, face_kind, face_u, F, eq):
    """One collide + stream step by an independent gather over explicit (x,y,z) triples, long double.
    f[(x,y,z)] -> list of Q values.  Written from Eq. 2/5, 6, 7, 10 and D:R6/R7, not from the oracle."""
    LD = np.longdouble
    nx, ny, nz = dims
    Q = len(E)
    post, rho_cell = {}, {}
    for c, fc in f.items():
        rho = sum(fc, LD(0))
        m = [sum((LD(E[a][d]) * fc[a] for a in range(Q)), LD(0)) for d in range(3)]
        div = rho if eq == EQ_STANDARD else LD(1)
        u = [(m[d] + LD(F[d]) / 2) / div for d in range(3)]
        usq = u[0] * u[0] + u[1] * u[1] + u[2] * u[2]
        out = []
        for a in range(Q):
            eu = E[a][0] * u[0] + E[a][1] * u[1] + E[a][2] * u[2]
            poly = 3 * eu + LD(9) / 2 * eu * eu - LD(3) / 2 * usq
            fe = LD(T[a]) * (rho * (1 + poly) if eq == EQ_STANDARD else rho + poly)
            src = sum(((3 * (E[a][d] - u[d]) + 9 * eu * E[a][d]) * LD(F[d]) for d in range(3)), LD(0))
            out.append(fc[a] - LD(omega) * (fc[a] - fe) + (1 - LD(omega) / 2) * LD(T[a]) * src)
        post[c] = out
        rho_cell[c] = rho if eq == EQ_STANDARD else LD(1)
    new = {}
    n = (nx, ny, nz)
    for c in f:
        vals = []
        for a in range(Q):
            src, wall, lid = [], False, -1
            for d in range(3):
                s = c[d] - E[a][d]
                if s < 0 or s >= n[d]:
                    face = 2 * d + (0 if s < 0 else 1)
                    if face_kind[face] == FACE_PERIODIC:
                        s %= n[d]
                    else:
                        wall = True
                        if face_kind[face] == FACE_MOVING:
                            lid = max(lid, face)
                src.append(s)
            if not wall:
                vals.append(post[tuple(src)][a])
            else:
                v = post[c][Q - 1 - a]
                if lid >= 0:
                    v = v + 6 * LD(T[a]) * rho_cell[c] * sum(E[a][d] * LD(face_u[lid][d]) for d in range(3))
                vals.append(v)
        new[c] = vals
    return new


_FACE_CASES = [
    ("periodic", [0] * 6, None),
    ("channel_z", [0, 0, 0, 0, 1, 1], None),
    ("cavity", [1, 1, 1, 1, 1, 2], {5: (0.1, 0.0, 0.0)}),
    ("mixed", [1, 2, 0, 0, 2, 1], {1: (0.0, 0.03, -0.02), 4: (0.05, 0.01, 0.0)}),
    ("all_moving", [2] * 6, {k: (0.01 * (k + 1), -0.02, 0.005 * k) for k in range(6)}),
]


@pytest.mark.parametrize("name,fk,fu", _FACE_CASES, ids=[c[0] for c in _FACE_CASES])
@pytest.mark.parametrize("Q,eq,forced", [(19, EQ_STANDARD, False), (19, EQ_STANDARD, True), (19, EQ_INCOMP, True),
                                         (27, EQ_STANDARD, True)])
def test_brute_force_small_grid(name, fk, fu, Q, eq, forced):
    """BASELINE.json north_star: '4^3 grids are brute-force-compared by hand-expanded updates' (here 4x5x4 so
    that a transposed axis cannot cancel), random non-equilibrium populations, 3 steps, every face-kind mix."""
    dims = (4, 5, 4)
    nx, ny, nz = dims
    N = nx * ny * nz
    if Q == 19:
        E = _E19
        T = [Fraction(1, 3) if sum(map(abs, v)) == 0 else Fraction(1, 18) if sum(map(abs, v)) == 1 else Fraction(1, 36) for v in E]
    else:
        E = list(itertools.product((-1, 0, 1), repeat=3))
        T = [[Fraction(8, 27), Fraction(2, 27), Fraction(1, 54), Fraction(1, 216)][sum(map(abs, v))] for v in E]
    Tld = [np.longdouble(t.numerator) / np.longdouble(t.denominator) for t in T]
    face_u = np.zeros((6, 3))
    for k, v in (fu or {}).items():
        face_u[k] = v
    F = (2e-4, -1e-4, 3e-4) if forced else (0.0, 0.0, 0.0)
    tau = 0.77
    rng = np.random.default_rng(42)
    f0 = np.array([float(t) for t in T])[:, None] * (1 + 0.2 * rng.uniform(-1, 1, (Q, N)))
    o = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=fk, face_u=face_u, force=F)
    o.set_f(f0)
    state = {}
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                i = x + nx * (y + ny * z)
                state[(x, y, z)] = [np.longdouble(f0[a, i]) for a in range(Q)]
    for _ in range(3):
        state = _brute_step(state, dims, E, Tld, np.longdouble(1) / np.longdouble(tau), fk, face_u, F, eq)
        o.step(1)
    got = o.get_f()
    ref = np.zeros_like(got)
    for (x, y, z), vals in state.items():
        ref[:, x + nx * (y + ny * z)] = [float(v) for v in vals]
    assert np.abs(got - ref).max() < 1e-15


def test_sweeps_are_the_papers_four(golden_dir):
    """step == Collision; BoundaryCondition; Propagation, and fb is the post-collision array."""
    n = 5
    rng = np.random.default_rng(7)
    _, w = lattice(19)
    f0 = w[:, None] * (1 + 0.1 * rng.standard_normal((19, n**3)))
    a = Oracle(n, n, n, 19, 0.6)
    b = Oracle(n, n, n, 19, 0.6)
    a.set_f(f0)
    b.set_f(f0)
    a.step(1)
    b.collision()
    b.boundary_condition()
    fb = b.get_fb().reshape(19, n, n, n)
    b.propagation()
    assert (a.get_f() == b.get_f()).all()
    # Eq. 7 on a periodic box: f_alpha(x) = fb_alpha(x - e_alpha)  <=>  roll fb by +e_alpha
    e, _ = lattice(19)
    f1 = b.get_f().reshape(19, n, n, n)  # [alpha, z, y, x]
    for q in range(19):
        assert (f1[q] == np.roll(fb[q], shift=(e[q, 2], e[q, 1], e[q, 0]), axis=(0, 1, 2))).all()


# ---------------------------------------------------------------------------- diagnostics (Monitor)
def _direct_diagnostics(f, act, E, F, eq):
    """The 8 diagnostics of include/lbm.h:161-166 evaluated from their definition on f[Q, N] (NumPy, no oracle code):
    { sum rho, sum rho u (3), 1/2 sum rho |u|^2, max |u|, min rho, non-finite cells } over the active nodes, non-finite
    cells excluded from the other seven; u = (sum e f + F/2) / rho (Eq. 8-9, D:R7), under Eq. 5 divided by and weighted
    with rho0 = 1 (D:R5); 3-component magnitude (D:R13)."""
    E = np.asarray(E, dtype=np.float64)
    with np.errstate(invalid="ignore", divide="ignore", over="ignore"):
        rho = f.sum(axis=0)
        m = E.T @ f + 0.5 * np.asarray(F, dtype=np.float64)[:, None]
        u = m / rho if eq == EQ_STANDARD else m.copy()
        usq = (u * u).sum(axis=0)
        ok = act.astype(bool) & np.isfinite(rho) & np.isfinite(usq)
    bad = int((act.astype(bool) & ~ok).sum())
    w = rho[ok] if eq == EQ_STANDARD else np.ones(int(ok.sum()))
    import math
    d = [math.fsum(rho[ok])] + [math.fsum(w * u[c][ok]) for c in range(3)]
    d += [0.5 * math.fsum(w * usq[ok]), float(np.sqrt(usq[ok]).max()), float(rho[ok].min()), float(bad)]
    return np.array(d), rho, u


@pytest.mark.parametrize("wall_model", [0, 1])
@pytest.mark.parametrize("Q,eq,forced", [(19, EQ_STANDARD, False), (19, EQ_STANDARD, True), (19, EQ_INCOMP, True),
                                         (27, EQ_STANDARD, True), (27, EQ_INCOMP, False), (9, EQ_STANDARD, True)])
def test_all_eight_diagnostics_equal_their_definition(Q, eq, forced, wall_model):
    """Every entry of post_processing's diagnostics[8] against a direct NumPy evaluation of its definition from the
    same populations: random non-equilibrium f, a solid mask (so inactive nodes exist and must be left out), both wall
    models, with and without the F/2 shift.  Catches a wrong constant (the 1/2 of the energy), a 2-component magnitude
    (P:415 as printed), rho vs rho0 weighting under Eq. 5, sums over inactive nodes."""
    if Q == 19:
        E = _E19
    else:
        E = [e for e in itertools.product((-1, 0, 1), repeat=3) if Q == 27 or e[2] == 0]
    dims = (9, 8, 7 if Q != 9 else 2)
    nx, ny, nz = dims
    N = nx * ny * nz
    F = (3e-3, -2e-3, 1e-3 if Q != 9 else 0.0) if forced else (0.0, 0.0, 0.0)
    o = Oracle(nx, ny, nz, Q, 0.7, eq=eq, force=F, face_kind=[FACE_PERIODIC] * 4 + ([FACE_BOUNCE] * 2 if Q != 9 else [FACE_PERIODIC] * 2))
    geo = np.zeros((nz, ny, nx), dtype=np.uint8)
    geo[: (4 if Q != 9 else nz), 2:6, 2:7] = 1  # a block on the z- wall: under the nodal model its skin becomes wall nodes, its core stays inactive
    o.set_geometry(geo.reshape(-1), wall_model)
    rng = np.random.default_rng(77 + Q + eq + wall_model)
    f0 = (1.0 / Q) * (1.0 + 0.4 * rng.uniform(-1, 1, (Q, N)))
    o.set_f(f0)
    f, act = o.get_f(), o.active()
    assert 0 < act.sum() < N
    rho_o, u_o, d_o = o.moments()
    d, rho, u = _direct_diagnostics(f, act, E, F, eq)
    np.testing.assert_allclose(d_o[:5], d[:5], rtol=1e-13, atol=1e-13)
    assert d_o[5] == pytest.approx(d[5], rel=1e-14) and d_o[6] == pytest.approx(d[6], rel=1e-14) and d_o[7] == d[7] == 0
    a = act.astype(bool)
    assert np.abs(rho_o[a] - rho[a]).max() <= 1e-14 and np.abs(u_o[:, a] - u[:, a]).max() <= 1e-14
    assert (rho_o[~a] == 0).all() and (u_o[:, ~a] == 0).all()
    # the energy really carries the factor 1/2 and all three components (not only its slope, as the Taylor-Green pin)
    assert d_o[4] == pytest.approx(0.5 * ((rho[a] if eq == EQ_STANDARD else 1.0) * (u[:, a] * u[:, a]).sum(axis=0)).sum(), rel=1e-12)


@pytest.mark.parametrize("eq", [EQ_STANDARD, EQ_INCOMP])
def test_nonfinite_cells_are_counted_and_left_out(eq):
    """One NaN and one Inf planted through set_f: diagnostics[7] = 2, the other seven finite and equal to the sums over
    the remaining cells (include/lbm.h: 'non-finite cells are excluded from the sums')."""
    nx, ny, nz, Q = 6, 5, 4, 19
    N = nx * ny * nz
    o = Oracle(nx, ny, nz, Q, 0.8, eq=eq, force=(1e-3, 0, 0))
    rng = np.random.default_rng(5)
    f0 = (1.0 / Q) * (1.0 + 0.3 * rng.uniform(-1, 1, (Q, N)))
    f0[3, 17] = np.nan
    f0[11, 60] = np.inf
    o.set_f(f0)
    _, _, d_o = o.moments()
    d, _, _ = _direct_diagnostics(f0, np.ones(N, dtype=np.uint8), _E19, (1e-3, 0, 0), eq)
    assert d_o[7] == 2 and d[7] == 2
    assert np.isfinite(d_o[:7]).all()
    np.testing.assert_allclose(d_o[:5], d[:5], rtol=1e-13, atol=1e-13)
    assert d_o[5] == pytest.approx(d[5], rel=1e-14) and d_o[6] == pytest.approx(d[6], rel=1e-14)
    clean = np.delete(f0, [17, 60], axis=1)
    assert d_o[0] == pytest.approx(clean.sum(), rel=1e-13)
