"""ctypes wrapper around oracle/liblbm_oracle.so (test infrastructure only).

All arrays are numpy float64 on the host, in the canonical layouts of include/lbm.h:
rho[i], u[c*N+i], f[alpha*N+i] with i = x + nx*(y + ny*z).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build

_lib = None

EQ_STANDARD, EQ_INCOMP = 0, 1
WALL_HALFWAY, WALL_NODAL = 0, 1
FACE_PERIODIC, FACE_BOUNCE, FACE_MOVING, FACE_PRESSURE, FACE_SYMMETRY = 0, 1, 2, 3, 4

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, _ip, _dp, _dp]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_lattice.argtypes = [C.c_int, _ip, _dp]
        lib.orc_feq.argtypes = [C.c_int, C.c_int, C.c_double, _dp, _dp]
        lib.orc_init_equilibrium.argtypes = [C.c_void_p, _dp, _dp]
        for name in ("orc_collision", "orc_boundary_condition", "orc_propagation"):
            getattr(lib, name).argtypes = [C.c_void_p]
        lib.orc_step.argtypes = [C.c_void_p, C.c_int]
        lib.orc_moments.argtypes = [C.c_void_p, _dp, _dp, _dp]
        for name in ("orc_get_f", "orc_get_fb", "orc_set_f"):
            getattr(lib, name).argtypes = [C.c_void_p, _dp]
        lib.orc_get_f_cells.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.c_int64, _dp]
        lib.orc_set_geometry.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        lib.orc_get_active.argtypes = [C.c_void_p, C.c_void_p]
        lib.orc_boundary_force.argtypes = [C.c_void_p, _dp]
        lib.orc_set_face_rho.argtypes = [C.c_void_p, _dp]
        lib.orc_set_face_velocity.argtypes = [C.c_void_p, C.c_int, _dp]
        lib.orc_num_threads.restype = C.c_int
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a, n):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64).reshape(-1)
    assert a.size == n, (a.size, n)
    return a


def num_threads() -> int:
    return int(_load().orc_num_threads())


def lattice(Q: int):
    """(e[Q,3] int, t[Q] float64) in the oracle's order."""
    e = np.zeros(3 * Q, dtype=np.int32)
    t = np.zeros(Q, dtype=np.float64)
    rc = _load().orc_lattice(Q, e.ctypes.data_as(_ip), _p(t))
    if rc != 0:
        raise ValueError(f"unknown lattice Q={Q}")
    return e.reshape(Q, 3), t


def feq(Q: int, eq: int, rho: float, u) -> np.ndarray:
    u = np.ascontiguousarray(u, dtype=np.float64)
    out = np.zeros(Q, dtype=np.float64)
    rc = _load().orc_feq(Q, eq, float(rho), _p(u), _p(out))
    if rc != 0:
        raise ValueError(f"unknown lattice Q={Q}")
    return out


class Oracle:
    def __init__(self, nx, ny, nz, Q=19, tau=0.8, eq=EQ_STANDARD, face_kind=None, face_u=None, force=None, face_rho=None):
        lib = _load()
        self.nx, self.ny, self.nz, self.Q = int(nx), int(ny), int(nz), int(Q)
        self.N = self.nx * self.ny * self.nz
        fk = np.zeros(6, dtype=np.int32) if face_kind is None else np.ascontiguousarray(face_kind, dtype=np.int32)
        fu = np.zeros((6, 3)) if face_u is None else np.ascontiguousarray(face_u, dtype=np.float64).reshape(6, 3)
        fo = np.zeros(3) if force is None else np.ascontiguousarray(force, dtype=np.float64).reshape(3)
        self._h = lib.orc_create(self.nx, self.ny, self.nz, self.Q, int(eq), float(tau),
                                 fk.ctypes.data_as(_ip), _p(fu), _p(fo))
        if not self._h:
            raise ValueError("orc_create failed (bad lattice, size or tau <= 0.5)")
        self._lib = lib
        if face_rho is not None:
            fr = np.ascontiguousarray(face_rho, dtype=np.float64).reshape(6)
            lib.orc_set_face_rho(self._h, _p(fr))

    def set_face_velocity(self, face, u=None):
        """Per-cell wall velocity of MOVING face `face`: u[3, n] over the face's cells (lower axis fastest); None = uniform."""
        uu = None if u is None else np.ascontiguousarray(u, dtype=np.float64).reshape(-1)
        if self._lib.orc_set_face_velocity(self._h, int(face), _p(uu)) != 0:
            raise ValueError("bad face")

    def close(self):
        if getattr(self, "_h", None):
            self._lib.orc_destroy(self._h)
            self._h = None

    __del__ = close

    def set_geometry(self, geo=None, wall_model=WALL_HALFWAY):
        """geo: N uint8 (non-zero = solid node) or None; call before init_equilibrium / set_f."""
        g = None if geo is None else np.ascontiguousarray(geo, dtype=np.uint8).reshape(-1)
        assert g is None or g.size == self.N
        rc = self._lib.orc_set_geometry(self._h, None if g is None else g.ctypes.data, int(wall_model))
        if rc != 0:
            raise ValueError("unknown wall model")

    def active(self):
        out = np.empty(self.N, dtype=np.uint8)
        self._lib.orc_get_active(self._h, out.ctypes.data)
        return out

    def boundary_force(self):
        F = np.empty(3)
        self._lib.orc_boundary_force(self._h, _p(F))
        return F

    def init_equilibrium(self, rho=None, u=None):
        rho, u = _f64(rho, self.N), _f64(u, 3 * self.N)
        self._lib.orc_init_equilibrium(self._h, _p(rho), _p(u))

    def collision(self):
        self._lib.orc_collision(self._h)

    def boundary_condition(self):
        self._lib.orc_boundary_condition(self._h)

    def propagation(self):
        self._lib.orc_propagation(self._h)

    def step(self, n=1):
        self._lib.orc_step(self._h, int(n))

    def moments(self, fields=True):
        rho = np.empty(self.N) if fields else None
        u = np.empty(3 * self.N) if fields else None
        diag = np.empty(8)
        self._lib.orc_moments(self._h, _p(rho), _p(u), _p(diag))
        return rho, (None if u is None else u.reshape(3, self.N)), diag

    def get_f(self):
        out = np.empty(self.Q * self.N)
        self._lib.orc_get_f(self._h, _p(out))
        return out.reshape(self.Q, self.N)

    def get_fb(self):
        out = np.empty(self.Q * self.N)
        self._lib.orc_get_fb(self._h, _p(out))
        return out.reshape(self.Q, self.N)

    def set_f(self, f):
        f = _f64(f, self.Q * self.N)
        self._lib.orc_set_f(self._h, _p(f))

    def get_f_cells(self, cells):
        cells = np.ascontiguousarray(cells, dtype=np.int64)
        out = np.empty((cells.size, self.Q))
        self._lib.orc_get_f_cells(self._h, cells.ctypes.data_as(C.POINTER(C.c_int64)), cells.size, _p(out))
        return out
