"""Pins for the geometry part of the CPU oracle (no GPU needed):
the solid mask `geo`, the paper's modified nodal bounce-back (Eq. 10)
and the momentum-exchange force (Eq. 13).  Each is checked against something other than
itself: the already-pinned face-built channel, an independent long-double gather on a tiny grid,
the paper's own accuracy claim ("second-order"), and the exact momentum balance of the fluid.

P:n = /root/reference/PAPER.md line n.  D:Rk = DESIGN.md reading k.
"""
import itertools
from fractions import Fraction

import numpy as np
import pytest

from oracle import Oracle
from oracle.binding import EQ_INCOMP, EQ_STANDARD, FACE_BOUNCE, FACE_PERIODIC, WALL_HALFWAY, WALL_NODAL

P_, B_ = FACE_PERIODIC, FACE_BOUNCE


def _lattice(Q):
    E = [v for v in itertools.product((-1, 0, 1), repeat=3) if Q == 27 or sum(map(abs, v)) < 3]
    w = {19: [Fraction(1, 3), Fraction(1, 18), Fraction(1, 36)],
         27: [Fraction(8, 27), Fraction(2, 27), Fraction(1, 54), Fraction(1, 216)]}[Q]
    return E, [w[sum(map(abs, v))] for v in E]


def _sphere(nx, ny, nz, c, r):
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return (((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2) <= r * r).astype(np.uint8).reshape(-1)


# --------------------------------------------------------------------------- the mask against the faces

@pytest.mark.parametrize("Q", [19, 27])
def test_mask_built_channel_equals_face_built_channel(Q):
    """Halfway walls: a z-periodic box whose planes z = 0 and z = H+1 are solid in `geo` is the same
    channel as an H-high box with BOUNCE faces at z-/z+ (pinned by the Poiseuille closed form in
    test_oracle_pins.py).  Same arithmetic per fluid node, so the populations agree bit for bit."""
    nx, ny, H = 5, 4, 6
    rng = np.random.default_rng(3)
    E, T = _lattice(Q)
    t = np.array([float(v) for v in T])
    f_in = t[:, None] * (1 + 0.2 * rng.uniform(-1, 1, (Q, nx * ny * H)))
    a = Oracle(nx, ny, H, Q, 0.7, face_kind=[P_, P_, P_, P_, B_, B_], force=(1e-4, 2e-4, 0))
    a.set_f(f_in)
    b = Oracle(nx, ny, H + 2, Q, 0.7, force=(1e-4, 2e-4, 0))
    geo = np.zeros((H + 2, ny, nx), dtype=np.uint8)
    geo[0] = geo[-1] = 1
    b.set_geometry(geo, WALL_HALFWAY)
    fb_in = np.zeros((Q, H + 2, ny * nx))
    fb_in[:, 1:-1] = f_in.reshape(Q, H, ny * nx)
    b.set_f(fb_in.reshape(Q, -1))
    a.step(7)
    b.step(7)
    fa = a.get_f().reshape(Q, H, ny * nx)
    fb = b.get_f().reshape(Q, H + 2, ny * nx)
    assert (fa == fb[:, 1:-1]).all()
    assert (fb[:, 0] == 0).all() and (fb[:, -1] == 0).all()  # inactive nodes report 0
    ra, ua, da = a.moments()
    rb, ub, db = b.moments()
    assert (ra.reshape(H, -1) == rb.reshape(H + 2, -1)[1:-1]).all()
    np.testing.assert_allclose(da[:5], db[:5], rtol=1e-14)  # sums run over the active nodes only
    assert da[5] == db[5] and da[6] == db[6]


def test_active_nodes_of_a_solid_cube():
    """D:R16: HALFWAY: active = fluid.  NODAL: plus the solid nodes with a fluid lattice neighbour — for a
    5^3 cube that is its one-node-thick shell (5^3 - 3^3 = 98 nodes), whichever lattice."""
    n = 9
    geo = np.zeros((n, n, n), dtype=np.uint8)
    geo[2:7, 2:7, 2:7] = 1
    for Q in (19, 27):
        o = Oracle(n, n, n, Q, 0.8)
        o.set_geometry(geo, WALL_HALFWAY)
        assert o.active().sum() == n**3 - 125
        o.set_geometry(geo, WALL_NODAL)
        act = o.active().reshape(n, n, n)
        assert act.sum() == n**3 - 125 + 98
        assert act[3:6, 3:6, 3:6].sum() == 0 and act[2, 2, 2] == 1


# --------------------------------------------------------------------------- brute force with a mask

def _brute_step_geo(f, active, dims, E, T, omega, periodic, F, eq, nodal):
    """One step by an independent gather over (x,y,z) triples in long double, written from Eq. 2/5, 6, 7, 10
    and D:R16/R17 (not from the oracle).  f: dict node -> list of Q values for the active nodes."""
    LD = np.longdouble
    Q = len(E)
    opp = [E.index(tuple(-c for c in v)) for v in E]

    def shift(c, a, sgn):
        out = []
        for d in range(3):
            s = c[d] + sgn * E[a][d]
            if s < 0 or s >= dims[d]:
                if not periodic[d]:
                    return None
                s %= dims[d]
            out.append(s)
        return tuple(out)

    post = {}
    for c, fc in f.items():
        rho = sum(fc, LD(0))
        m = [sum((LD(E[a][d]) * fc[a] for a in range(Q)), LD(0)) for d in range(3)]
        div = rho if eq == EQ_STANDARD else LD(1)
        u = [(m[d] + LD(F[d]) / 2) / div for d in range(3)]
        usq = sum(v * v for v in u)
        out = []
        for a in range(Q):
            eu = sum(E[a][d] * u[d] for d in range(3))
            poly = 3 * eu + LD(9) / 2 * eu * eu - LD(3) / 2 * usq
            fe = LD(T[a]) * (rho * (1 + poly) if eq == EQ_STANDARD else rho + poly)
            src = sum(((3 * (E[a][d] - u[d]) + 9 * eu * E[a][d]) * LD(F[d]) for d in range(3)), LD(0))
            out.append(fc[a] - LD(omega) * (fc[a] - fe) + (1 - LD(omega) / 2) * LD(T[a]) * src)
        post[c] = out
    new = {}
    for c in f:
        vals, unknown = [None] * Q, []
        for a in range(Q):
            up = shift(c, a, -1)
            if up is not None and up in active:
                vals[a] = post[up][a]
            elif not nodal:
                vals[a] = post[c][opp[a]]  # halfway bounce-back
            else:
                unknown.append(a)
        for a in unknown:  # Eq. 10 after propagation
            dn = shift(c, a, +1)
            vals[a] = vals[opp[a]] if (dn is not None and dn in active) else post[c][opp[a]]
        new[c] = vals
    return new


@pytest.mark.parametrize("nodal", [False, True], ids=["halfway", "nodal"])
@pytest.mark.parametrize("Q,eq,faces", [(19, EQ_STANDARD, [P_] * 6), (27, EQ_STANDARD, [B_, B_, P_, P_, B_, B_]),
                                        (19, EQ_INCOMP, [P_, P_, B_, B_, P_, P_])])
def test_brute_force_with_mask(nodal, Q, eq, faces):
    dims = (6, 7, 6)
    nx, ny, nz = dims
    N = nx * ny * nz
    E, T = _lattice(Q)
    Tld = [np.longdouble(t.numerator) / np.longdouble(t.denominator) for t in T]
    geo = np.zeros((nz, ny, nx), dtype=np.uint8)
    geo[1:5, 2:6, 1:4] = 1  # a 3x4x4 block (thick enough to have an inactive core under NODAL)
    geo[5, 0, 5] = 1        # and a single solid node next to a corner
    F = (2e-4, -1e-4, 3e-4)
    tau = 0.77
    o = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=faces, force=F)
    o.set_geometry(geo, WALL_NODAL if nodal else WALL_HALFWAY)
    # independent activity classification
    periodic = [faces[0] == P_, faces[2] == P_, faces[4] == P_]
    solid = {(x, y, z) for z in range(nz) for y in range(ny) for x in range(nx) if geo[z, y, x]}
    active = set()
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                c = (x, y, z)
                if c not in solid:
                    active.add(c)
                elif nodal:
                    for v in E:
                        nb, ok = [], True
                        for d in range(3):
                            s = c[d] + v[d]
                            if s < 0 or s >= dims[d]:
                                if not periodic[d]:
                                    ok = False
                                    break
                                s %= dims[d]
                            nb.append(s)
                        if ok and tuple(nb) not in solid:
                            active.add(c)
                            break
    act = o.active().reshape(nz, ny, nx)
    assert {(x, y, z) for z in range(nz) for y in range(ny) for x in range(nx) if act[z, y, x]} == active
    rng = np.random.default_rng(5)
    f0 = np.array([float(t) for t in T])[:, None] * (1 + 0.2 * rng.uniform(-1, 1, (Q, N)))
    o.set_f(f0)
    f0 = o.get_f()  # D:R17: the state is made consistent with Eq. 10 (nodal) and inactive nodes report 0
    state = {c: [np.longdouble(f0[a, c[0] + nx * (c[1] + ny * c[2])]) for a in range(Q)] for c in active}
    for _ in range(3):
        state = _brute_step_geo(state, active, dims, E, Tld, np.longdouble(1) / np.longdouble(tau), periodic, F, eq, nodal)
        o.step(1)
    got = o.get_f()
    ref = np.zeros_like(got)
    for (x, y, z), vals in state.items():
        ref[:, x + nx * (y + ny * z)] = [float(v) for v in vals]
    assert np.abs(got - ref).max() < 1e-15


def test_nodal_state_is_consistent_with_eq10_at_time_zero():
    """D:R17: after init, a wall node's unknown directions already hold their opposites (Eq. 10)."""
    nx, ny, nz = 3, 3, 6
    o = Oracle(nx, ny, nz, 19, 0.8, face_kind=[P_, P_, P_, P_, B_, B_])
    o.set_geometry(None, WALL_NODAL)
    u = np.zeros((3, nx * ny * nz))
    u[0] = 0.03
    u[2] = 0.02
    o.init_equilibrium(None, u)
    f = o.get_f().reshape(19, nz, ny * nx)
    E, _ = _lattice(19)
    for a, v in enumerate(E):
        if v[2] == 1:   # nothing streams into the bottom wall nodes along +z
            assert (f[a, 0] == f[18 - a, 0]).all()
        if v[2] == -1:
            assert (f[a, -1] == f[18 - a, -1]).all()
    # interior nodes are the plain equilibrium
    assert np.ptp(f[:, 2], axis=1).max() == 0


# --------------------------------------------------------------------------- nodal bounce-back: accuracy

def _nodal_channel_error(nz, Q, tau=0.9, Fx=1e-6):
    """Forced channel between nodal walls on the planes z = 0 and z = nz-1 (width H = nz-1), run to steady state."""
    H = nz - 1
    nu = (tau - 0.5) / 3
    o = Oracle(1, 1, nz, Q, tau, face_kind=[P_, P_, P_, P_, B_, B_], force=(Fx, 0, 0))
    o.set_geometry(None, WALL_NODAL)
    o.init_equilibrium(None, None)
    o.step(int(40 * H * H / (np.pi**2 * nu)))
    _, u, d = o.moments()
    z = np.arange(nz, dtype=float)
    ref = Fx * z * (H - z) / (2 * nu)
    assert abs(d[0] - nz) / nz < 1e-9  # Eq. 10 copies populations, so mass is only conserved up to the transient
    return np.abs(u[0] - ref).max() / ref.max(), u[0]


@pytest.mark.parametrize("Q", [19, 27])
def test_nodal_bounce_back_is_second_order(Q):
    """'second-order modified nodal bounce back'.  The steady channel profile converges to the parabola
    through the WALL NODES (wall on the node, D:R3) with an error that falls 4x per doubling of the width."""
    e8, u8 = _nodal_channel_error(9, Q)
    e16, _ = _nodal_channel_error(17, Q)
    e32, _ = _nodal_channel_error(33, Q)
    assert e8 < 0.05 and e16 < e8 and e32 < e16
    assert 3.5 < e8 / e16 < 4.5 and 3.5 < e16 / e32 < 4.5
    assert np.abs(u8 - u8[::-1]).max() < 1e-15 * 1e6  # mirror symmetry of the profile (u ~ 1e-5)


def test_halfway_and_nodal_walls_sit_where_they_should():
    """Wall placement (D:R3): with the same 16 active planes the halfway channel is 16 wide (walls half a link
    outside) and the nodal one 15 wide (walls on the first and last plane), so the centreline velocities differ
    by about (16/15)^2."""
    tau, Fx, nz = 0.9, 1e-6, 16
    nu = (tau - 0.5) / 3
    res = []
    for model in (WALL_HALFWAY, WALL_NODAL):
        o = Oracle(1, 1, nz, 19, tau, face_kind=[P_, P_, P_, P_, B_, B_], force=(Fx, 0, 0))
        o.set_geometry(None, model)
        o.init_equilibrium(None, None)
        o.step(30000)
        res.append(o.moments()[1][0].max())
    assert res[0] / (Fx * 16**2 / (8 * nu)) == pytest.approx(1.0, abs=0.01)
    assert res[1] / (Fx * 15**2 / (8 * nu)) == pytest.approx(1.0, abs=0.02)


# --------------------------------------------------------------------------- momentum exchange (Eq. 13)

@pytest.mark.parametrize("model", [WALL_HALFWAY, WALL_NODAL], ids=["halfway", "nodal"])
@pytest.mark.parametrize("Q", [19, 27])
def test_momentum_exchange_balances_fluid_momentum(Q, model):
    """Eq. 13 against the exact momentum balance of the fluid region R (geo = 0) in a periodic box with a
    sphere and a body force:  sum_R e f (t+1) - sum_R e f (t) = |R| F - F_wall.  The left side comes from the
    moment fields only (rho u = sum e f + F/2), i.e. not from the code that evaluates Eq. 13."""
    n = 14
    Fb = np.array([3e-5, -1e-5, 2e-5])
    geo = _sphere(n, n, n, (6.3, 7.1, 6.6), 3.6)
    fluid = geo == 0
    o = Oracle(n, n, n, Q, 0.8, force=Fb)
    o.set_geometry(geo, model)
    rng = np.random.default_rng(1)
    o.init_equilibrium(1 + 0.01 * rng.standard_normal(n**3), 0.02 * rng.standard_normal((3, n**3)))

    def momentum():
        rho, u, _ = o.moments()
        return np.array([(rho[fluid] * u[c][fluid]).sum() for c in range(3)])

    o.step(3)
    for _ in range(4):
        m0 = momentum()
        o.step(1)
        m1 = momentum()
        Fw = o.boundary_force()
        np.testing.assert_allclose(fluid.sum() * Fb - (m1 - m0), Fw, rtol=0, atol=1e-13 * np.abs(Fw).max() + 1e-15)
        assert np.abs(Fw).max() > 1e-6  # the sphere really exchanges momentum with this noisy flow


def test_steady_drag_equals_total_body_force():
    """At steady state the body (halfway walls) carries exactly the force fed into the fluid: F_wall = |R| F."""
    n = 12
    Fb = np.array([1e-5, 0, 0])
    geo = _sphere(n, n, n, (5.5, 5.5, 5.5), 2.7)
    o = Oracle(n, n, n, 19, 1.0, force=Fb)
    o.set_geometry(geo, WALL_HALFWAY)
    o.init_equilibrium(None, None)
    o.step(4000)
    Fw = o.boundary_force()
    assert Fw[0] == pytest.approx((geo == 0).sum() * Fb[0], rel=1e-6)
    assert abs(Fw[1]) < 1e-12 and abs(Fw[2]) < 1e-12
