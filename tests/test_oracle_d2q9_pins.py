"""Pins for the oracle's D2Q9 path (CPU only).  The table itself is pinned to the
paper's printed Eq. 3-4 in test_oracle_pins.py; here the dynamics on that table are checked against things other
than the oracle: 2-D isotropy identities, equilibrium moments, an independent brute-force gather in long double,
the exact 2-D Taylor-Green decay (second-order convergence), the Poiseuille closed form with halfway walls, and
exact conservation.  P:n = /root/reference/PAPER.md line n.
"""
import itertools
from fractions import Fraction

import numpy as np
import pytest

from oracle import Oracle, feq, lattice
from oracle.binding import EQ_INCOMP, EQ_STANDARD, FACE_BOUNCE, FACE_MOVING, FACE_PERIODIC
from paper_2201_11330_b200 import inputs

P_, B_, M_ = FACE_PERIODIC, FACE_BOUNCE, FACE_MOVING


def test_d2q9_isotropy_in_two_dimensions():
    """Eq. 3-4 satisfy the 2-D moment identities with c_s^2 = 1/3 up to order 5."""
    e, w = lattice(9)
    assert (e[:, 2] == 0).all()
    e = e[:, :2].astype(float)
    d = np.eye(2)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs(np.einsum("q,qi->i", w, e)).max() < 1e-16
    np.testing.assert_allclose(np.einsum("q,qi,qj->ij", w, e, e), d / 3, atol=1e-16)
    assert np.abs(np.einsum("q,qi,qj,qk->ijk", w, e, e, e)).max() < 1e-16
    iso4 = (np.einsum("ij,kl->ijkl", d, d) + np.einsum("ik,jl->ijkl", d, d) + np.einsum("il,jk->ijkl", d, d)) / 9
    np.testing.assert_allclose(np.einsum("q,qi,qj,qk,ql->ijkl", w, e, e, e, e), iso4, atol=1e-16)
    assert np.abs(np.einsum("q,qi,qj,qk,ql,qm->ijklm", w, e, e, e, e, e)).max() < 1e-16


@pytest.mark.parametrize("eq", [EQ_STANDARD, EQ_INCOMP])
def test_d2q9_equilibrium_moments(eq):
    """Eq. 2 / Eq. 5 on D2Q9: sum feq = rho, sum e feq = A u, sum e e feq = rho/3 I + A u u (A = rho or rho0 = 1)."""
    e, _ = lattice(9)
    e = e[:, :2].astype(float)
    rng = np.random.default_rng(4)
    for _ in range(5):
        rho = 1 + 0.1 * rng.standard_normal()
        u = np.append(0.1 * rng.standard_normal(2), 0.0)
        A = rho if eq == EQ_STANDARD else 1.0
        fe = feq(9, eq, rho, u)
        assert abs(fe.sum() - rho) < 1e-15
        np.testing.assert_allclose(fe @ e, A * u[:2], atol=1e-16)
        np.testing.assert_allclose(np.einsum("q,qi,qj->ij", fe, e, e), rho / 3 * np.eye(2) + A * np.outer(u[:2], u[:2]), atol=1e-16)


def _brute_step_2d(f, dims, omega, faces, face_u, F, eq):
    """One step written from Eq. 2/5, 6, 7, 10 and D:R6/R7 with a hand-typed D2Q9 table (the paper's Eq. 3-4),
    as a gather over explicit (x, y) pairs in long double.  f: [9, ny, nx]."""
    LD = np.longdouble
    E = [(-1, -1), (-1, 0), (-1, 1), (0, -1), (0, 0), (0, 1), (1, -1), (1, 0), (1, 1)]
    T = [Fraction(1, 36), Fraction(1, 9), Fraction(1, 36), Fraction(1, 9), Fraction(4, 9), Fraction(1, 9), Fraction(1, 36),
         Fraction(1, 9), Fraction(1, 36)]
    T = [LD(t.numerator) / LD(t.denominator) for t in T]
    nx, ny = dims
    post = np.zeros((9, ny, nx), dtype=LD)
    rho_all = np.zeros((ny, nx), dtype=LD)
    for y, x in itertools.product(range(ny), range(nx)):
        fc = f[:, y, x]
        rho = sum(fc, LD(0))
        m = [sum((LD(E[a][d]) * fc[a] for a in range(9)), LD(0)) for d in range(2)]
        div = rho if eq == EQ_STANDARD else LD(1)
        u = [(m[d] + LD(F[d]) / 2) / div for d in range(2)]
        usq = u[0] * u[0] + u[1] * u[1]
        rho_all[y, x] = rho if eq == EQ_STANDARD else LD(1)
        for a in range(9):
            eu = E[a][0] * u[0] + E[a][1] * u[1]
            poly = 3 * eu + LD(9) / 2 * eu * eu - LD(3) / 2 * usq
            fe = T[a] * (rho * (1 + poly) if eq == EQ_STANDARD else rho + poly)
            src = sum(((3 * (E[a][d] - u[d]) + 9 * eu * E[a][d]) * LD(F[d]) for d in range(2)), LD(0))
            post[a, y, x] = fc[a] - LD(omega) * (fc[a] - fe) + (1 - LD(omega) / 2) * T[a] * src
    new = np.zeros_like(post)
    n = (nx, ny)
    for y, x in itertools.product(range(ny), range(nx)):
        c = (x, y)
        for a in range(9):
            up, inside, mface = [], True, -1
            for d in range(2):
                s = c[d] - E[a][d]
                if s < 0 or s >= n[d]:
                    face = 2 * d + (0 if s < 0 else 1)
                    if faces[face] == P_:
                        s %= n[d]
                    else:
                        inside = False
                        if faces[face] == M_:
                            mface = max(mface, face)
                up.append(s)
            if inside:
                new[a, y, x] = post[a, up[1], up[0]]
            else:
                v = post[8 - a, y, x]
                if mface >= 0:
                    v += 6 * T[a] * rho_all[y, x] * (E[a][0] * LD(face_u[mface][0]) + E[a][1] * LD(face_u[mface][1]))
                new[a, y, x] = v
    return new


@pytest.mark.parametrize("eq", [EQ_STANDARD, EQ_INCOMP])
@pytest.mark.parametrize("faces", [[P_, P_, P_, P_], [B_, B_, P_, P_], [B_, M_, M_, B_]])
def test_d2q9_brute_force(eq, faces):
    nx, ny = 5, 4
    rng = np.random.default_rng(9)
    f0 = (1.0 / 9) * (1 + 0.2 * rng.uniform(-1, 1, (9, ny * nx)))
    face_u = np.zeros((6, 3))
    face_u[1] = (0.0, 0.04, 0.0)
    face_u[2] = (0.03, 0.0, 0.0)
    F = (2e-4, -1e-4, 0.0)
    tau = 0.77
    o = Oracle(nx, ny, 1, 9, tau, eq=eq, face_kind=faces + [P_, P_], face_u=face_u, force=F)
    o.set_f(f0)
    state = f0.reshape(9, ny, nx).astype(np.longdouble)
    for _ in range(3):
        state = _brute_step_2d(state, (nx, ny), np.longdouble(1) / np.longdouble(tau), faces, face_u, F, eq)
        o.step(1)
    assert np.abs(o.get_f() - state.reshape(9, -1).astype(float)).max() < 1e-15


def _tgv2d_rate_error(n, tau=0.8, u0=0.01):
    rho, u = inputs.taylor_green_2d(n, n, 1, u0)
    o = Oracle(n, n, 1, 9, tau)
    o.init_equilibrium(rho, u)
    nu, k2 = (tau - 0.5) / 3, 2 * (2 * np.pi / n) ** 2
    steps = int(round(0.5 / (nu * k2)))
    o.step(steps // 4)  # let the initial layer of the equilibrium start die out
    a0 = np.abs(o.moments()[1][0]).max()
    o.step(steps)
    a1 = np.abs(o.moments()[1][0]).max()
    return -np.log(a1 / a0) / steps / (nu * k2) - 1


def test_d2q9_taylor_green_decay_is_second_order():
    """2-D Taylor-Green vortex (exact Navier-Stokes solution): the velocity decays as exp(-nu |k|^2 t), nu = (tau-1/2)/3
    (D:R1), |k|^2 = 2 (2 pi/n)^2; the rate error falls ~4x per doubling of n."""
    e16, e32, e64 = (abs(_tgv2d_rate_error(n)) for n in (16, 32, 64))
    assert e16 < 1e-2 and e32 < 2.5e-3 and e64 < 7e-4
    assert 3.0 < e16 / e32 < 5.0 and 3.0 < e32 / e64 < 5.0


def test_d2q9_conserves_mass_and_momentum():
    n = 24
    rho, u = inputs.taylor_green_2d(n, n, 1, 0.05)
    rho = rho + inputs.density_noise(n, n, 1, 1e-3, 7) - 1
    o = Oracle(n, n, 1, 9, 0.6)
    o.init_equilibrium(rho, u)
    d0 = o.moments(False)[2]
    o.step(200)
    d1 = o.moments(False)[2]
    assert abs(d1[0] - d0[0]) / d0[0] < 1e-13
    np.testing.assert_allclose(d1[1:4], d0[1:4], atol=1e-12)


def test_d2q9_poiseuille_closed_form():
    """Body-forced channel between halfway walls on D2Q9: u(y) = F/(2 nu) [ y (H - y) + 4 Lambda/3 - 1/4 ],
    Lambda = (tau - 1/2)^2, y = k + 1/2 (the parabola plus the BGK wall-slip constant), to 1e-9."""
    H, tau, F = 12, 0.9, 1e-6
    nu = (tau - 0.5) / 3
    o = Oracle(1, H, 1, 9, tau, face_kind=[P_, P_, B_, B_, P_, P_], force=(F, 0, 0))
    o.init_equilibrium(None, None)
    o.step(6000)
    ux = o.moments()[1][0]
    y = np.arange(H) + 0.5
    ref = F / (2 * nu) * (y * (H - y) + 4 * (tau - 0.5) ** 2 / 3 - 0.25)
    assert np.abs(ux - ref).max() / ref.max() < 1e-9


def test_d2q9_planes_do_not_talk():
    """With nz > 1 the D2Q9 planes are independent copies (e_z = 0)."""
    nx, ny, nz = 6, 5, 3
    rng = np.random.default_rng(2)
    f0 = (1.0 / 9) * (1 + 0.2 * rng.uniform(-1, 1, (9, nz, ny * nx)))
    o = Oracle(nx, ny, nz, 9, 0.7)
    o.set_f(f0.reshape(9, -1))
    o.step(4)
    got = o.get_f().reshape(9, nz, ny * nx)
    for k in range(nz):
        one = Oracle(nx, ny, 1, 9, 0.7)
        one.set_f(f0[:, k].copy())
        one.step(4)
        assert (one.get_f() == got[:, k]).all()
