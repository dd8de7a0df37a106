"""Host logic of the seeded input recipes (paper_2201_11330_b200/inputs.py) — no GPU, no LBM
arithmetic: the workloads that stand in for the paper's examples carry the parameters the paper prints, sub-boxes are
generated point-wise, and reduced copies keep the physics.  The oracle runs the reduced examples for a few steps to show
that every recipe is a well-posed input (finite, mass-conserving where it must be)."""
import os

import numpy as np
import pytest

from oracle import Oracle
from paper_2201_11330_b200 import inputs


def _oracle_of(w):
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force, face_rho=w.face_rho)
    if w.has_geometry:
        o.set_geometry(w.geo(), w.wall_model)
    for k, prof in w.face_profiles().items():
        o.set_face_velocity(k, prof)
    return o


def test_channel_cylinder_recipes_carry_the_papers_numbers(golden_dir):
    """tests/golden/paper_drag.txt quotes P:439-462; configs 6 and 7 must be those cases."""
    rows = {}
    with open(os.path.join(golden_dir, "paper_drag.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, nx, ny, D, cx, om, Re, cd = line.split()
                rows[k] = (int(nx), int(ny), float(D), float(cx), float(om), float(Re))
    for case, cfg in (("case1", 6), ("case2", 7)):
        nx, ny, D, cx, om, Re = rows[case]
        w = inputs.config(cfg)
        assert (w.nx, w.ny, w.nz, w.Q) == (nx, ny, 1, 9)
        assert w.cylinder == (cx, (ny - 1) / 2.0, D / 2.0)
        assert abs(1.0 / w.tau - om) < 1e-12
        nu = (w.tau - 0.5) / 3.0                       # DESIGN.md R1
        assert abs(w.inlet_umax * D / nu - Re) < 1e-9  # R23: U = centreline inlet velocity
        assert w.face_kind == (inputs.FACE_MOVING, inputs.FACE_PRESSURE, inputs.FACE_BOUNCE, inputs.FACE_BOUNCE, 0, 0)
        prof = w.face_profiles()[0]
        assert prof.shape == (3, ny) and prof[1:].max() == 0.0
        # parabola between the halfway walls: symmetric, zero at the walls (y = -1/2, ny - 1/2), maximum U on the centreline
        assert np.allclose(prof[0], prof[0][::-1])
        assert abs(prof[0].max() - w.inlet_umax * (1 - 1.0 / ny**2)) < 1e-15
        y = np.arange(ny) + 0.5
        assert np.allclose(prof[0], w.inlet_umax * 4 * y * (ny - y) / ny**2)
        geo = w.geo().reshape(ny, nx)
        assert geo.sum() == pytest.approx(np.pi * (D / 2) ** 2, rel=0.03)  # a disc of diameter D
        assert (geo == geo[::-1]).all()                                    # centred between the walls


def test_sphere_case_recipes():
    """512 x 128 x 128, sphere r = 8 at (64,64,64), D3Q27; config 8 adds the boundaries the paper names."""
    for cfg in (5, 8):
        w = inputs.config(cfg)
        assert (w.nx, w.ny, w.nz, w.Q) == (512, 128, 128, 27) and w.sphere == (64.0, 64.0, 64.0, 8.0)
        assert w.wall_model == inputs.WALL_NODAL and w.eq == inputs.EQ_INCOMP
    w = inputs.config(8)
    S = inputs.FACE_SYMMETRY
    assert w.face_kind == (inputs.FACE_MOVING, inputs.FACE_PRESSURE, S, S, 0, 0) and w.force == (0.0, 0.0, 0.0)
    small = w.shrunk(8)
    g = small.geo()
    assert g.sum() == 7 and g.reshape(16, 16, 64)[8, 8, 8] == 1  # radius-1 sphere: centre + 6 neighbours


def test_sub_boxes_are_generated_point_wise():
    """Any sub-box of a config equals the same region of the full field (used by the sampled 512^3 parity tests and by
    the z-slab halo planes), periodic wrap included."""
    for cfg in (0, 7):
        w = inputs.config(cfg).shrunk(2) if cfg == 7 else inputs.config(cfg)
        rho, u = w.fields()
        nz = w.nz
        box = ((3, 9), (w.ny - 2, w.ny + 3), (0, 1) if nz == 1 else (nz - 1, nz + 2))
        r2, u2 = w.fields(box=box)
        xs = np.arange(*box[0]) % w.nx
        ys = np.arange(*box[1]) % w.ny
        zs = np.arange(*box[2]) % w.nz
        idx = (xs[None, None, :] + w.nx * (ys[None, :, None] + w.ny * zs[:, None, None])).reshape(-1)
        assert np.array_equal(r2, rho[idx]) and np.array_equal(u2, u[:, idx])


@pytest.mark.parametrize("cfg,k,steps", [(7, 4, 300), (8, 4, 100), (5, 8, 60)])
def test_reduced_examples_are_well_posed(cfg, k, steps):
    """The oracle on reduced copies of the paper's examples: finite, near-incompressible, drag pointing downstream."""
    w = inputs.config(cfg).shrunk(k, steps=steps)
    rho, u = w.fields()
    o = _oracle_of(w)
    o.init_equilibrium(rho, u)
    o.step(w.steps)
    r, v, d = o.moments()
    act = o.active().astype(bool)
    assert d[7] == 0 and np.isfinite(r).all() and np.isfinite(v).all()
    assert np.abs(r[act] - 1.0).max() < 0.05 and d[5] < 0.2
    if w.kind in ("channel", "inflow"):  # an oncoming stream pushes the body downstream from the start
        assert o.boundary_force()[0] > 0.0
    o.close()
