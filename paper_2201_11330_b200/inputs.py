"""Seeded synthetic inputs for the BASELINE.json configs (numpy only).

This module holds NO lattice-Boltzmann arithmetic: it only produces the macroscopic
initial fields (rho, u) and the boundary description that are handed, unchanged, to both
the CUDA library and the CPU oracle.  It imports neither of them.

Recipe:
  * Taylor-Green vortex on a 2*pi box with x_i = 2*pi*i/n:
        u = u0 * ( sin x cos y cos z, -cos x sin y cos z, 0 )
  * density noise rho = 1 + a*(2r - 1), r in [0,1) from a counter-based hash of
    (seed, global cell index) so that any sub-box can be generated point-wise.
Layouts: rho[i], u[c*N + i], i = x + nx*(y + ny*z).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

SEED_BASE = 0x22011330

FACE_PERIODIC, FACE_BOUNCE, FACE_MOVING, FACE_PRESSURE, FACE_SYMMETRY = 0, 1, 2, 3, 4
EQ_STANDARD, EQ_INCOMP = 0, 1
WALL_HALFWAY, WALL_NODAL = 0, 1

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def hash_uniform(seed: int, index: np.ndarray) -> np.ndarray:
    """Counter-based uniform r in [0,1): splitmix64 finaliser of (seed, index), top 53 bits."""
    with np.errstate(over="ignore"):
        z = index.astype(np.uint64) + np.uint64(seed & 0xFFFFFFFFFFFFFFFF) * np.uint64(0x9E3779B97F4A7C15)
        z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _axes(n, lo, hi, wrap):
    """Global integer coordinates lo..hi-1 of one axis, wrapped into [0, n) if asked."""
    g = np.arange(lo, hi, dtype=np.int64)
    return np.mod(g, n) if wrap else g


def taylor_green(nx, ny, nz, u0, noise=0.0, seed=0, box=None):
    """rho[N], u[3,N] of the 3-D Taylor-Green vortex (+ seeded density noise).

    `box` = ((x0,x1),(y0,y1),(z0,z1)) evaluates the SAME global field on a sub-box whose
    coordinates are wrapped periodically into the global grid (for sampled parity checks).
    """
    if box is None:
        box = ((0, nx), (0, ny), (0, nz))
    gx = _axes(nx, *box[0], True)
    gy = _axes(ny, *box[1], True)
    gz = _axes(nz, *box[2], True)
    X = 2.0 * np.pi * gx / nx
    Y = 2.0 * np.pi * gy / ny
    Z = 2.0 * np.pi * gz / nz
    sx, cx = np.sin(X)[None, None, :], np.cos(X)[None, None, :]
    sy, cy = np.sin(Y)[None, :, None], np.cos(Y)[None, :, None]
    cz = np.cos(Z)[:, None, None]
    n = gx.size * gy.size * gz.size
    u = np.zeros((3, n))
    u[0] = (u0 * sx * cy * cz).reshape(-1)
    u[1] = (-u0 * cx * sy * cz).reshape(-1)
    rho = density_noise(nx, ny, nz, noise, seed, box)
    return rho, u


def taylor_green_2d(nx, ny, nz, u0):
    """z-invariant 2-D Taylor-Green vortex with its exact pressure field.

    u = u0 (sin x cos y, -cos x sin y, 0),  rho = 1 + 3 (u0^2/4)(cos 2x + cos 2y)
    (p = rho/3): an exact Navier-Stokes solution decaying as exp(-2 nu k^2 t) per velocity
    component, |k|^2 = 2 (2 pi/n)^2 (SURVEY.md section 8c pins).
    """
    X = 2.0 * np.pi * np.arange(nx) / nx
    Y = 2.0 * np.pi * np.arange(ny) / ny
    sx, cx = np.sin(X)[None, None, :], np.cos(X)[None, None, :]
    sy, cy = np.sin(Y)[None, :, None], np.cos(Y)[None, :, None]
    one = np.ones((nz, 1, 1))
    n = nx * ny * nz
    u = np.zeros((3, n))
    u[0] = (u0 * sx * cy * one).reshape(-1)
    u[1] = (-u0 * cx * sy * one).reshape(-1)
    rho = (1.0 + 3.0 * (u0 * u0 / 4.0) * (np.cos(2 * X)[None, None, :] + np.cos(2 * Y)[None, :, None]) * one).reshape(-1)
    return rho, u


def density_noise(nx, ny, nz, noise, seed, box=None):
    """rho = 1 + noise*(2r-1) on the whole grid or on a (periodically wrapped) sub-box."""
    if box is None:
        box = ((0, nx), (0, ny), (0, nz))
    gx = _axes(nx, *box[0], True)
    gy = _axes(ny, *box[1], True)
    gz = _axes(nz, *box[2], True)
    n = gx.size * gy.size * gz.size
    if noise == 0.0:
        return np.ones(n)
    gi = (gx[None, None, :] + nx * (gy[None, :, None] + ny * gz[:, None, None])).reshape(-1)
    return 1.0 + noise * (2.0 * hash_uniform(seed, gi) - 1.0)


def sphere_mask(nx, ny, nz, centre, radius):
    """uint8[N]: 1 where (x-cx)^2 + (y-cy)^2 + (z-cz)^2 <= r^2 (lattice nodes inside or on the sphere)."""
    x = np.arange(nx)[None, None, :] - centre[0]
    y = np.arange(ny)[None, :, None] - centre[1]
    z = np.arange(nz)[:, None, None] - centre[2]
    return ((x * x + y * y + z * z) <= radius * radius).astype(np.uint8).reshape(-1)


def cylinder_mask(nx, ny, nz, centre, radius):
    """uint8[N]: 1 where (x-cx)^2 + (y-cy)^2 <= r^2 — a z-invariant circular cylinder (Fig. 3)."""
    x = np.arange(nx)[None, None, :] - centre[0]
    y = np.arange(ny)[None, :, None] - centre[1]
    m = ((x * x + y * y) <= radius * radius) & np.ones((nz, 1, 1), dtype=bool)
    return m.astype(np.uint8).reshape(-1)


def parabola(n, umax):
    """Poiseuille profile between halfway walls at -1/2 and n-1/2: umax * 4 (k+1/2)(n-k-1/2)/n^2, k = 0..n-1."""
    k = np.arange(n) + 0.5
    return umax * 4.0 * k * (n - k) / (n * n)


@dataclass
class Workload:
    """One BASELINE.json config: geometry, physics parameters and how to make its fields."""
    name: str
    nx: int
    ny: int
    nz: int
    Q: int
    tau: float
    steps: int
    face_kind: tuple = (0, 0, 0, 0, 0, 0)
    face_u: tuple = field(default_factory=lambda: tuple((0.0, 0.0, 0.0) for _ in range(6)))
    force: tuple = (0.0, 0.0, 0.0)
    u0: float = 0.0
    noise: float = 0.0
    seed: int = 0
    kind: str = "tgv"  # "tgv" | "rest" | "channel" (parabolic inflow) | "inflow" (uniform inflow)
    eq: int = EQ_STANDARD
    wall_model: int = WALL_HALFWAY
    sphere: tuple | None = None  # (cx, cy, cz, r): nodes with |x - c| <= r are solid
    cylinder: tuple | None = None  # (cx, cy, r): z-invariant circular cylinder
    face_rho: tuple | None = None  # density prescribed on FACE_PRESSURE faces (6 values)
    inlet_umax: float = 0.0  # "channel": parabolic profile u_x(y) on the x- MOVING face and as the initial field

    @property
    def N(self):
        return self.nx * self.ny * self.nz

    @property
    def has_geometry(self):
        return self.sphere is not None or self.cylinder is not None or self.wall_model != WALL_HALFWAY

    def geo(self):
        """Solid mask (uint8[N], 1 = solid node; the paper's `geo`) or None."""
        if self.sphere is not None:
            return sphere_mask(self.nx, self.ny, self.nz, self.sphere[:3], self.sphere[3])
        if self.cylinder is not None:
            return cylinder_mask(self.nx, self.ny, self.nz, self.cylinder[:2], self.cylinder[2])
        return None

    def face_profiles(self):
        """{face: u[3, n]} per-cell wall velocities of MOVING faces (lower in-face axis fastest); {} = uniform."""
        if self.kind != "channel":
            return {}
        prof = np.zeros((3, self.ny * self.nz))
        prof[0] = np.tile(parabola(self.ny, self.inlet_umax), self.nz)  # j = y + ny*z
        return {0: prof}

    def shrunk(self, k, steps=None):
        """Same workload with every length (grid, sphere, cylinder) divided by k."""
        sp = None if self.sphere is None else tuple(v / k for v in self.sphere)
        # node j sits at j + 1/2 between the halfway walls: scale that position, not the index
        cy = None if self.cylinder is None else ((self.cylinder[0] + 0.5) / k - 0.5, (self.cylinder[1] + 0.5) / k - 0.5, self.cylinder[2] / k)
        return replace(self, name=f"{self.name}/{k}", nx=self.nx // k, ny=self.ny // k, nz=max(1, self.nz // k),
                       steps=steps or self.steps, sphere=sp, cylinder=cy)

    def fields(self, box=None):
        """(rho[n], u[3,n]) on the full grid or on a periodically wrapped sub-box."""
        if self.kind == "tgv":
            return taylor_green(self.nx, self.ny, self.nz, self.u0, self.noise, self.seed, box)
        rho = density_noise(self.nx, self.ny, self.nz, self.noise, self.seed, box)
        u = np.zeros((3, rho.size))
        if self.kind == "inflow":
            u[0] = self.inlet_umax  # the uniform inflow velocity everywhere
        if self.kind == "channel":
            # the inlet profile at every x ("steady-state inviscid flow with randomly distributed perturbation")
            b = box or ((0, self.nx), (0, self.ny), (0, self.nz))
            gy = _axes(self.ny, *b[1], True)
            ux = parabola(self.ny, self.inlet_umax)[gy]
            u[0] = np.broadcast_to(ux[None, :, None], (b[2][1] - b[2][0], gy.size, b[0][1] - b[0][0])).reshape(-1)
        return rho, u

    def scaled(self, n, steps=None, name=None):
        """Same parameters on an n^3 grid (reduced analogue for oracle-affordable parity)."""
        sp = None if self.sphere is None else tuple(v * n / self.ny for v in self.sphere)
        return replace(self, name=name or f"{self.name}@{n}", nx=n, ny=n, nz=n, steps=steps or self.steps, sphere=sp)


_CAVITY_FACES = (FACE_BOUNCE,) * 5 + (FACE_MOVING,)
_LID_U = tuple((0.0, 0.0, 0.0) for _ in range(5)) + ((0.1, 0.0, 0.0),)
_CHANNEL_FACES = (FACE_PERIODIC,) * 4 + (FACE_BOUNCE, FACE_BOUNCE)


def config(i: int) -> Workload:
    """BASELINE.json configs[i], i = 0..4 (file order); 5 = the paper's sphere case (S:§8f NEXT-2)."""
    if i == 0:
        return Workload("cfg0_q19_tgv32", 32, 32, 32, 19, 0.8, 100, u0=0.05, noise=1e-4, seed=SEED_BASE + 1)
    if i == 1:
        return Workload("cfg1_q19_tgv128", 128, 128, 128, 19, 0.6, 1000, u0=0.05, noise=1e-4, seed=SEED_BASE + 2)
    if i == 2:
        return Workload("cfg2_q19_cavity256", 256, 256, 256, 19, 0.55, 2000, face_kind=_CAVITY_FACES,
                        face_u=_LID_U, kind="rest")
    if i == 3:
        return Workload("cfg3_q19_tgv512", 512, 512, 512, 19, 0.52, 200, u0=0.04, noise=1e-4, seed=SEED_BASE + 4)
    if i == 4:
        return Workload("cfg4_q27_channel512", 512, 512, 512, 27, 0.9, 20000, face_kind=_CHANNEL_FACES,
                        force=(1e-7, 0.0, 0.0), noise=1e-5, seed=SEED_BASE + 5, kind="rest")
    if i == 5:
        # Not in BASELINE.json: the paper's own profiled / validated case — D3Q27, 512 x 128 x 128,
        # sphere of radius 8 at (64,64,64), the incompressible model the paper's code runs (Eq. 5) with its nodal
        # bounce-back on the sphere.  The inlet / outlet / symmetric sides have no formulae in the paper, so the
        # box is periodic and the flow is driven by a body force.
        return Workload("cfg5_q27_sphere512x128x128", 512, 128, 128, 27, 1.0 / 1.8, 6401, force=(1e-6, 0.0, 0.0),
                        noise=1e-5, seed=SEED_BASE + 6, kind="rest", eq=EQ_INCOMP, wall_model=WALL_NODAL,
                        sphere=(64.0, 64.0, 64.0, 8.0))
    if i in (6, 7):
        # Not in BASELINE.json: the paper's 2-D channel-cylinder example (section 4), D2Q9, Eq. 5 model.
        #   case 1 (i = 6): 1024 x 1024, D = 32, centre 512 from the inlet, omega = 1.8,   Re = U D / nu = 20  (C_D -> 2.06)
        #   case 2 (i = 7):  512 x  128, D = 16, centre  64 from the inlet, omega = 1.953, Re = 100            (C_D ~ 1.46)
        # Inlet = parabolic velocity profile on x- (MOVING + per-cell wall velocity), outlet = PRESSURE rho = 1 on x+,
        # no-slip BOUNCE walls on y-, y+ (R22: the paper gives no formulae for its inlet / outflow); U = the
        # centreline inlet velocity (R23).  The cylinder is a solid mask with halfway bounce-back.
        nx, ny, D, cx, omega, Re, steps = ((1024, 1024, 32.0, 512.0, 1.8, 20.0, 200000) if i == 6
                                           else (512, 128, 16.0, 64.0, 1.953, 100.0, 100000))
        tau = 1.0 / omega
        nu = (tau - 0.5) / 3.0
        U = Re * nu / D
        return Workload(f"cfg{i}_q9_cylinder{nx}x{ny}", nx, ny, 1, 9, tau, steps,
                        face_kind=(FACE_MOVING, FACE_PRESSURE, FACE_BOUNCE, FACE_BOUNCE, FACE_PERIODIC, FACE_PERIODIC),
                        noise=1e-5, seed=SEED_BASE + i + 1, kind="channel", eq=EQ_INCOMP,
                        cylinder=(cx, (ny - 1) / 2.0, D / 2.0), face_rho=(1.0,) * 6, inlet_umax=U)
    if i == 8:
        # Not in BASELINE.json: the paper's sphere case with the boundaries P:468 names — "the back surface is inlet and
        # the front surface is outlet, the left and right boundaries are symmetric, and the top and bottom boundaries
        # are periodic": x- MOVING (uniform inflow U), x+ PRESSURE rho = 1, y-/y+ SYMMETRY, z periodic (R22,
        # R24, R25); D3Q27, Eq. 5, nodal bounce-back on the sphere as in config 5.  U = 0.05 (Re = U D / nu = 43).
        U = 0.05
        return Workload("cfg8_q27_sphere_open512x128x128", 512, 128, 128, 27, 1.0 / 1.8, 6401,
                        face_kind=(FACE_MOVING, FACE_PRESSURE, FACE_SYMMETRY, FACE_SYMMETRY, FACE_PERIODIC, FACE_PERIODIC),
                        face_u=((U, 0.0, 0.0),) + tuple((0.0, 0.0, 0.0) for _ in range(5)),
                        noise=1e-5, seed=SEED_BASE + 9, kind="inflow", eq=EQ_INCOMP, wall_model=WALL_NODAL,
                        sphere=(64.0, 64.0, 64.0, 8.0), face_rho=(1.0,) * 6, inlet_umax=U)
    raise IndexError(i)
