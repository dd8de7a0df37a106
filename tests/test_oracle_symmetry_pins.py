"""Pins of the oracle's SYMMETRY faces (R25: "the left and right boundaries are symmetric", no
formula) and of open faces next to the paper's nodal wall model (R24).  Pinned by what the mathematics fixes:

  * a mirror plane is, by definition, equivalent to the mirror-extended domain: the same flow computed on the
    doubled box (which uses only already-pinned features: periodic wrap, bounce-back, masks, nodal walls, open
    faces) must reproduce the half box — for one symmetric face, for two (doubled box periodic), for an edge where
    two symmetry planes meet, with a solid mask touching the plane, under both wall models;
  * free slip: a uniform flow along a symmetry plane stays exactly uniform (no wall friction), and a channel with
    one wall and one symmetry plane has the Poiseuille profile of the channel of twice the height;
  * an independent long-double gather written here from the rules of R6 / R16 / R17 / R22 / R24 / R25 over every
    mix of face kinds with a mask and both wall models.

P:n = /root/reference/PAPER.md line n.
"""
import numpy as np
import pytest

from oracle import Oracle
from typed_lattice import typed_lattice
from oracle.binding import EQ_INCOMP, EQ_STANDARD, WALL_HALFWAY, WALL_NODAL

P, B, M, PR, S = 0, 1, 2, 3, 4
LD = np.longdouble


def _flip_table(E, axis):
    """a -> index of e_a with component `axis` negated."""
    E = [tuple(int(v) for v in row) for row in E]
    return [E.index(tuple(-v if d == axis else v for d, v in enumerate(e))) for e in E]


# --------------------------------------------------------------------------- mirror-extended domain
def _mirror_extend(arr, axis_np):
    """[..., nz, ny, nx] -> doubled along axis_np: mirror image first, then the original (plane between them)."""
    return np.concatenate([np.flip(arr, axis=axis_np), arr], axis=axis_np)


def _run_pair(dims, Q, eq, model, fk, doubled_axes, steps, geo=None, tau=0.63, seed=0, face_u=None, face_rho=None):
    """Half box with SYMMETRY on the lower face of every axis in doubled_axes (and on the upper one too if the
    face list says so) against the mirror-extended box.  Returns max |f_half - f_doubled restricted|."""
    nx, ny, nz = dims
    E, T = typed_lattice(Q)  # typed by hand (tests/typed_lattice.py), not the oracle's own table
    rng = np.random.default_rng(seed)
    f0 = T[:, None, None, None] * (1.0 + 0.2 * rng.uniform(-1, 1, (Q, nz, ny, nx)))
    g0 = np.zeros((nz, ny, nx), dtype=np.uint8) if geo is None else geo.reshape(nz, ny, nx)
    half = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=fk, face_u=face_u, face_rho=face_rho)
    half.set_geometry(g0, model)
    half.set_f(f0.reshape(Q, -1))

    fd, gd, fkd, dd = f0, g0, list(fk), [nx, ny, nz]
    for ax in doubled_axes:          # ax: 0 = x, 1 = y, 2 = z
        npax = 3 - ax                # axis of f0[Q, z, y, x]
        flip = _flip_table(E, ax)
        img = np.flip(fd, axis=npax)[flip]  # the image node carries the mirrored direction (flip is an involution)
        fd = np.concatenate([img, fd], axis=npax)
        gd = _mirror_extend(gd, npax - 1)
        dd[ax] *= 2
        lo, hi = fk[2 * ax], fk[2 * ax + 1]
        assert lo == S
        # lower face of the doubled box = mirror image of the upper face; both symmetric -> the doubled box is periodic
        fkd[2 * ax], fkd[2 * ax + 1] = (P, P) if hi == S else (hi, hi)
    full = Oracle(dd[0], dd[1], dd[2], Q, tau, eq=eq, face_kind=fkd, face_u=face_u, face_rho=face_rho)
    full.set_geometry(gd, model)
    full.set_f(fd.reshape(Q, -1))
    half.step(steps)
    full.step(steps)
    fh = half.get_f().reshape(Q, nz, ny, nx)
    ff = full.get_f().reshape(Q, dd[2], dd[1], dd[0])
    sl = [slice(None)] * 4
    for ax in doubled_axes:
        n = dims[ax]
        sl[3 - ax] = slice(n, 2 * n)
    err = float(np.abs(fh - ff[tuple(sl)]).max())
    rh = half.moments()[0]
    half.close()
    full.close()
    return err, rh


def _blob(dims, touch_axis):
    """A solid lump that touches the lower face of touch_axis (so the mirror plane cuts a body) + a free one."""
    nx, ny, nz = dims
    g = np.zeros((nz, ny, nx), dtype=np.uint8)
    idx = [slice(nz // 2 - 1, nz // 2 + 1), slice(ny // 2 - 1, ny // 2 + 1), slice(nx // 2 - 1, nx // 2 + 1)]
    idx[2 - touch_axis] = slice(0, 2)
    g[tuple(idx)] = 1
    g[nz - 2, ny - 2, nx - 2] = 1
    return g


@pytest.mark.parametrize("model", [WALL_HALFWAY, WALL_NODAL], ids=["halfway", "nodal"])
@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_INCOMP)])
@pytest.mark.parametrize("name,fk,axes", [
    ("sym_ylo_wall_yhi", [P, P, S, B, P, P], [1]),
    ("sym_both_y", [P, P, S, S, P, P], [1]),
    ("sym_edge_y_z", [P, P, S, S, S, B], [1, 2]),
    ("sym_xlo_walls", [S, B, B, B, P, P], [0]),
])
def test_symmetry_face_equals_mirror_extended_domain(name, fk, axes, Q, eq, model):
    dims = (6, 5, 6)
    err, _ = _run_pair(dims, Q, eq, model, fk, axes, steps=6, geo=_blob(dims, axes[0]), seed=3)
    assert err <= 1e-14, (name, err)


def test_symmetry_d2q9_with_open_faces():
    """D2Q9 channel half: inlet (uniform, along x), pressure outlet, wall at y+, mirror plane at y-: equals the full
    channel of twice the height.  The inlet velocity has no component normal to the mirror."""
    fk = [M, PR, S, B, P, P]
    fu = np.zeros((6, 3))
    fu[0] = (0.04, 0.0, 0.0)
    err, _ = _run_pair((9, 6, 1), 9, EQ_INCOMP, WALL_HALFWAY, fk, [1], steps=8, seed=5, face_u=fu,
                       face_rho=[1, 0.98, 1, 1, 1, 1])
    assert err <= 1e-14, err


# --------------------------------------------------------------------------- free slip
@pytest.mark.parametrize("Q", [9, 19, 27])
def test_uniform_flow_along_symmetry_planes_is_preserved(Q):
    """No friction on a mirror plane: u = (U,0,0) between two symmetry planes (periodic in x) is a steady state."""
    nz = 1 if Q == 9 else 4
    fk = [P, P, S, S, P, P] if Q == 9 else [P, P, S, S, S, S]
    o = Oracle(6, 5, nz, Q, 0.7, face_kind=fk)
    N = 6 * 5 * nz
    u = np.zeros((3, N))
    u[0] = 0.05
    o.init_equilibrium(None, u)
    f0 = o.get_f().copy()
    o.step(50)
    assert np.abs(o.get_f() - f0).max() <= 1e-15
    o.close()


def test_half_channel_has_the_profile_of_the_full_channel():
    """Wall at z-, mirror plane at z+ (H = 8) and a body force: steady u(z) is the Poiseuille parabola of the channel
    of height 2H, u(z) = F/(2 nu) [ z (2H - z) + 4 Lambda/3 - 1/4 ], z = k + 1/2 (parabola + BGK halfway-wall slip)."""
    H, tau, F = 8, 0.9, 1e-6
    nu = (tau - 0.5) / 3.0
    o = Oracle(3, 3, H, 19, tau, face_kind=[P, P, P, P, B, S], force=(F, 0, 0))
    o.init_equilibrium()
    o.step(12000)
    u = o.moments()[1][0].reshape(H, 9).mean(axis=1)
    z = np.arange(H) + 0.5
    ref = F / (2 * nu) * (z * (2 * H - z) + 4.0 * (tau - 0.5) ** 2 / 3.0 - 0.25)
    assert np.abs(u - ref).max() <= 1e-9 * ref.max()
    o.close()


# --------------------------------------------------------------------------- brute force over every rule at once
def _profile_index(face, c, dims):
    nx, ny, nz = dims
    x, y, z = c
    return [y + ny * z, y + ny * z, x + nx * z, x + nx * z, x + nx * y, x + nx * y][face]


def _brute_step(f, active, dims, E, T, omega, fk, fu, prof, frho, eq, nodal, F):
    """One collide + stream step in long double on dicts of nodes, written from Eq. 2/5, 6, 7, 10 and the readings
    R6 (Ladd), R7 (Guo), R16/R17 (active nodes, Eq. 10), R22 (open faces), R24 (open faces next to nodal walls),
    R25 (mirror planes) — not from the oracle."""
    Q = len(E)
    opp = [E.index(tuple(-v for v in e)) for e in E]
    post, rho_c, u_c = {}, {}, {}
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
        post[c], rho_c[c], u_c[c] = out, (rho if eq == EQ_STANDARD else LD(1)), u

    def source(c, a, sgn):
        """('node', node, direction) | ('moving', face) | ('pressure', face) | ('wall',) for the link of node c along
        sgn * e_a."""
        node, e2, crossed = [], list(E[a]), []
        for d in range(3):
            s = c[d] + sgn * E[a][d]
            if s < 0 or s >= dims[d]:
                face = 2 * d + (0 if s < 0 else 1)
                if fk[face] == P:
                    s %= dims[d]
                else:
                    crossed.append(face)
                    if fk[face] == S:
                        s, e2[d] = c[d], -e2[d]
            node.append(s)
        kinds = [fk[k] for k in crossed]
        if M in kinds:
            return ("moving", max(k for k in crossed if fk[k] == M))
        if B in kinds:
            return ("wall",)
        if PR in kinds:
            return ("pressure", max(k for k in crossed if fk[k] == PR))
        node = tuple(node)
        return ("node", node, E.index(tuple(e2))) if node in active else ("wall",)

    new = {}
    for c in f:
        vals, unknown = [None] * Q, []
        for a in range(Q):
            src = source(c, a, -1)
            if src[0] == "node":
                vals[a] = post[src[1]][src[2]]
            elif src[0] == "moving":
                k = src[1]
                uw = [LD(prof[k][d][_profile_index(k, c, dims)]) for d in range(3)] if k in prof else [LD(fu[k][d]) for d in range(3)]
                vals[a] = post[c][opp[a]] + 6 * LD(T[a]) * rho_c[c] * sum(E[a][d] * uw[d] for d in range(3))
            elif src[0] == "pressure":
                u = u_c[c]
                eu = sum(E[a][d] * u[d] for d in range(3))
                even = LD(9) / 2 * eu * eu - LD(3) / 2 * sum(x * x for x in u)
                rf = LD(frho[src[1]])
                vals[a] = -post[c][opp[a]] + 2 * LD(T[a]) * (rf * (1 + even) if eq == EQ_STANDARD else rf + even)
            elif not nodal:
                vals[a] = post[c][opp[a]]
            else:
                unknown.append(a)
        for a in unknown:  # Eq. 10 after propagation (R17)
            vals[a] = vals[opp[a]] if source(c, a, +1)[0] == "node" else post[c][opp[a]]
        new[c] = vals
    return new


_MIXES = [
    ("sphere_case_faces", [M, PR, S, S, P, P]),        # inlet, outlet, symmetric sides, periodic top / bottom
    ("duct_sym_walls", [M, PR, S, B, B, S]),
    ("all_kinds", [S, PR, M, B, PR, S]),
    ("sym_everywhere", [S] * 6),
    ("inlet_outlet_walls", [M, PR, B, B, P, P]),       # the channel-cylinder faces, R24 under the nodal model
]


@pytest.mark.parametrize("nodal", [False, True], ids=["halfway", "nodal"])
@pytest.mark.parametrize("Q,eq", [(19, EQ_STANDARD), (27, EQ_INCOMP), (9, EQ_INCOMP)])
@pytest.mark.parametrize("name,fk", _MIXES, ids=[m[0] for m in _MIXES])
def test_brute_force_all_face_kinds_with_mask(name, fk, Q, eq, nodal):
    dims = (5, 4, 1) if Q == 9 else (5, 4, 4)
    nx, ny, nz = dims
    N = nx * ny * nz
    fk = list(fk)
    if Q == 9:
        fk[4] = fk[5] = P
    E, T = typed_lattice(Q)  # typed by hand (tests/typed_lattice.py), not the oracle's own table
    E = [tuple(int(v) for v in row) for row in E]
    rng = np.random.default_rng(17 + Q)
    f0 = T[:, None] * (1.0 + 0.2 * rng.uniform(-1, 1, (Q, N)))
    fu = np.zeros((6, 3))
    frho = np.array([1.0, 0.97, 1.02, 0.99, 1.01, 0.98])
    prof = {}
    for k in range(6):
        if fk[k] == M:
            fu[k] = (0.01 * (k + 1), -0.015, 0.004 * k)
            if k % 4 == 0:
                prof[k] = 0.03 * rng.uniform(-1, 1, (3, [ny * nz, ny * nz, nx * nz, nx * nz, nx * ny, nx * ny][k]))
    geo = np.zeros((nz, ny, nx), dtype=np.uint8)
    geo[nz // 2, 1:3, 2] = 1   # a two-node body in the interior
    geo[0, 0, 0] = 1           # a solid corner node: touches three faces at once
    geo[nz - 1, ny - 1, 1:3] = 1
    force = (1e-4, -2e-4, 0.0)
    tau = 0.71
    o = Oracle(nx, ny, nz, Q, tau, eq=eq, face_kind=fk, face_u=fu, face_rho=frho, force=force)
    for k, pr in prof.items():
        o.set_face_velocity(k, pr)
    o.set_geometry(geo, WALL_NODAL if nodal else WALL_HALFWAY)
    act = o.active().reshape(nz, ny, nx)
    o.set_f(f0)
    got0 = o.get_f()  # under the nodal model set_f makes the state consistent with Eq. 10; start the brute force from it
    cells = [(x, y, z) for z in range(nz) for y in range(ny) for x in range(nx) if act[z, y, x]]
    f = {c: [LD(got0[a, c[0] + nx * (c[1] + ny * c[2])]) for a in range(Q)] for c in cells}
    active = set(cells)
    for _ in range(3):
        f = _brute_step(f, active, dims, E, T, 1.0 / tau, fk, fu, prof, frho, eq, nodal, force)
    o.step(3)
    got = o.get_f()
    o.close()
    for c in cells:
        i = c[0] + nx * (c[1] + ny * c[2])
        ref = np.array([float(v) for v in f[c]])
        assert np.abs(got[:, i] - ref).max() <= 2e-15, (name, c)
