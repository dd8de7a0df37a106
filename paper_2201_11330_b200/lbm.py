"""Thin ctypes binding over the C ABI of include/lbm.h (same names, argument marshalling only).

Every step of the path runs in the CUDA library; torch is used for device memory, streams
and events.  There is no CPU fallback: if the library cannot be loaded, `load()` raises.

Functions mirror the C names one to one (`lbm_create`, `lbm_init_equilibrium`, `lbm_step`,
`lbm_moments`, ...).  `Solver` is a small convenience wrapper that owns a handle.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

LBM_D2Q9, LBM_D3Q19, LBM_D3Q27 = 9, 19, 27
LBM_EQ_STANDARD, LBM_EQ_INCOMP = 0, 1 << 8
LBM_SCHEME_AUTO, LBM_SCHEME_AB, LBM_SCHEME_AA = 0, 1 << 12, 2 << 12
LBM_STORE_F64, LBM_STORE_F32 = 0, 1 << 16
LBM_LAYOUT_ROWS, LBM_LAYOUT_SOA = 0, 1 << 20
LBM_FACE_PERIODIC, LBM_FACE_BOUNCE, LBM_FACE_MOVING, LBM_FACE_PRESSURE, LBM_FACE_SYMMETRY = 0, 1, 2, 3, 4
LBM_WALL_HALFWAY, LBM_WALL_NODAL = 0, 1
LBM_OK, LBM_EINVAL, LBM_ENOMEM, LBM_ECUDA, LBM_EUNSUPPORTED = 0, -1, -2, -3, -4
LBM_STATIC_MAX_CELLS = 1 << 27  # largest grid lbm_diagnostics_static accepts (its scratch array is fixed)

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "liblbm_b200.so")

# every symbol include/lbm.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "lbm_create", "lbm_destroy", "lbm_init_equilibrium", "lbm_init_equilibrium_host", "lbm_step",
    "lbm_moments", "lbm_moments_host", "lbm_get_populations", "lbm_set_populations", "lbm_lattice",
    "lbm_time", "lbm_launch_count", "lbm_set_block", "lbm_set_persistent", "lbm_set_two_step", "lbm_last_error",
    "lbm_set_geometry", "lbm_set_geometry_host", "lbm_boundary_force",
    "lbm_set_face_velocity", "lbm_set_face_velocity_host", "lbm_set_face_density",
    "lbm_create_slab", "lbm_slab_export", "lbm_slab_connect", "lbm_slab_set_sync",
    "lbm_debug_arm", "lbm_debug_check", "lbm_diagnostics_static",
)


class lbm_bc_t(C.Structure):
    _fields_ = [
        ("face_kind", C.c_int32 * 6),
        ("face_u", (C.c_double * 3) * 6),
        ("force", C.c_double * 3),
        ("stream", C.c_void_p),
    ]


class lbm_slab_peer_t(C.Structure):
    """What a neighbouring z-slab needs to know about a slab (include/lbm.h); plain bytes, picklable via bytes()."""
    _fields_ = [
        ("buf", C.c_uint64 * 2),
        ("flags", C.c_uint64),
        ("plane_stride", C.c_int64),
        ("nz_local", C.c_int32),
        ("device", C.c_int32),
        ("pid", C.c_int64),
        ("Q", C.c_int32),
        ("elem_bytes", C.c_int32),
        ("layout_soa", C.c_int32),
        ("reserved", C.c_int32),
        ("stream", C.c_uint64),
        ("ipc_buf", (C.c_uint8 * 64) * 2),
        ("ipc_flags", C.c_uint8 * 64),
    ]


class LBMError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"lbm error {code}: {msg}")
        self.code = code


_lib = None


def load():
    """Load liblbm_b200.so (built in-tree by `python -m paper_2201_11330_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2201_11330_b200.build` "
            "(the CUDA library is the only implementation; there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp, i32, i64 = C.c_void_p, C.c_void_p, C.c_int, C.c_int64
    lib.lbm_create.restype = vp
    lib.lbm_create.argtypes = [i32, i32, i32, i32, C.c_double, C.POINTER(lbm_bc_t)]
    lib.lbm_destroy.restype = None
    lib.lbm_destroy.argtypes = [vp]
    for name in ("lbm_init_equilibrium", "lbm_init_equilibrium_host"):
        getattr(lib, name).restype = i32
        getattr(lib, name).argtypes = [vp, dp, dp]
    lib.lbm_step.restype = i32
    lib.lbm_step.argtypes = [vp, i32]
    for name in ("lbm_moments", "lbm_moments_host"):
        getattr(lib, name).restype = i32
        getattr(lib, name).argtypes = [vp, dp, dp, dp]
    for name in ("lbm_get_populations", "lbm_set_populations"):
        getattr(lib, name).restype = i32
        getattr(lib, name).argtypes = [vp, dp]
    lib.lbm_lattice.restype = i32
    lib.lbm_lattice.argtypes = [i32, C.POINTER(C.c_int32), C.POINTER(C.c_double)]
    lib.lbm_time.restype = i64
    lib.lbm_time.argtypes = [vp]
    lib.lbm_launch_count.restype = i64
    lib.lbm_launch_count.argtypes = [vp]
    lib.lbm_set_block.restype = i32
    lib.lbm_set_block.argtypes = [vp, i32, i32]
    lib.lbm_set_persistent.restype = i32
    lib.lbm_set_persistent.argtypes = [vp, i32]
    lib.lbm_set_two_step.restype = i32
    lib.lbm_set_two_step.argtypes = [vp, i32]
    for name in ("lbm_set_geometry", "lbm_set_geometry_host"):
        getattr(lib, name).restype = i32
        getattr(lib, name).argtypes = [vp, C.c_void_p, i32]
    lib.lbm_boundary_force.restype = i32
    lib.lbm_boundary_force.argtypes = [vp, C.c_void_p]
    for name in ("lbm_set_face_velocity", "lbm_set_face_velocity_host"):
        getattr(lib, name).restype = i32
        getattr(lib, name).argtypes = [vp, i32, dp]
    lib.lbm_set_face_density.restype = i32
    lib.lbm_set_face_density.argtypes = [vp, C.c_void_p]
    lib.lbm_create_slab.restype = vp
    lib.lbm_create_slab.argtypes = [i32, i32, i32, i32, i32, i32, C.c_double, C.POINTER(lbm_bc_t)]
    lib.lbm_slab_export.restype = i32
    lib.lbm_slab_export.argtypes = [vp, C.POINTER(lbm_slab_peer_t)]
    lib.lbm_slab_connect.restype = i32
    lib.lbm_slab_connect.argtypes = [vp, C.POINTER(lbm_slab_peer_t), C.POINTER(lbm_slab_peer_t)]
    lib.lbm_slab_set_sync.restype = i32
    lib.lbm_slab_set_sync.argtypes = [vp, i32]
    lib.lbm_debug_arm.restype = i32
    lib.lbm_debug_arm.argtypes = [vp, i32]
    lib.lbm_debug_check.restype = i64
    lib.lbm_debug_check.argtypes = [vp]
    lib.lbm_diagnostics_static.restype = i32
    lib.lbm_diagnostics_static.argtypes = [dp, i64, i32, C.c_void_p, dp, vp]
    lib.lbm_last_error.restype = C.c_char_p
    lib.lbm_last_error.argtypes = []
    _lib = lib
    return lib


def lbm_last_error() -> str:
    return load().lbm_last_error().decode()


def _check(rc):
    if rc != 0:
        raise LBMError(rc, lbm_last_error())


def _ptr(t, n=None, device="cuda"):
    """Raw address of a contiguous float64 torch tensor (or None)."""
    if t is None:
        return None
    import torch
    assert isinstance(t, torch.Tensor) and t.dtype == torch.float64 and t.is_contiguous(), "need a contiguous float64 tensor"
    assert t.device.type == device, f"tensor must live on {device}, got {t.device}"
    assert n is None or t.numel() == n, (t.numel(), n)
    return t.data_ptr()


def make_bc(face_kind=None, face_u=None, force=None, stream=None) -> lbm_bc_t:
    bc = lbm_bc_t()
    fk = [0] * 6 if face_kind is None else list(face_kind)
    fu = np.zeros((6, 3)) if face_u is None else np.asarray(face_u, dtype=np.float64).reshape(6, 3)
    fo = np.zeros(3) if force is None else np.asarray(force, dtype=np.float64).reshape(3)
    for k in range(6):
        bc.face_kind[k] = int(fk[k])
        for d in range(3):
            bc.face_u[k][d] = float(fu[k, d])
    for d in range(3):
        bc.force[d] = float(fo[d])
    bc.stream = None if stream is None else int(stream)
    return bc


# ---- one function per C entry point ----------------------------------------------------
def lbm_create(nx, ny, nz, lattice, tau, bc: lbm_bc_t | None = None):
    h = load().lbm_create(int(nx), int(ny), int(nz), int(lattice), float(tau), None if bc is None else C.byref(bc))
    if not h:
        raise LBMError(LBM_EINVAL, lbm_last_error())
    return h


def lbm_destroy(h):
    load().lbm_destroy(h)


def lbm_create_slab(nx, ny, nz_local, z0, nz_global, lattice, tau, bc: lbm_bc_t | None = None):
    h = load().lbm_create_slab(int(nx), int(ny), int(nz_local), int(z0), int(nz_global), int(lattice), float(tau),
                               None if bc is None else C.byref(bc))
    if not h:
        raise LBMError(LBM_EINVAL, lbm_last_error())
    return h


def lbm_slab_export(h) -> lbm_slab_peer_t:
    d = lbm_slab_peer_t()
    _check(load().lbm_slab_export(h, C.byref(d)))
    return d


def lbm_slab_connect(h, lower: lbm_slab_peer_t | None, upper: lbm_slab_peer_t | None):
    _check(load().lbm_slab_connect(h, None if lower is None else C.byref(lower), None if upper is None else C.byref(upper)))


def lbm_slab_set_sync(h, device_sync: bool):
    _check(load().lbm_slab_set_sync(h, 1 if device_sync else 0))


def _u8ptr(t, n, device):
    if t is None:
        return None
    import torch
    assert isinstance(t, torch.Tensor) and t.dtype == torch.uint8 and t.is_contiguous(), "need a contiguous uint8 tensor"
    assert t.device.type == device and t.numel() == n, (t.device, t.numel(), n)
    return t.data_ptr()


def lbm_set_geometry(h, geo, wall_model, n):
    """geo: uint8 CUDA tensor of n = N bytes (non-zero = solid) or None."""
    _check(load().lbm_set_geometry(h, _u8ptr(geo, n, "cuda"), int(wall_model)))


def lbm_set_geometry_host(h, geo, wall_model, n):
    _check(load().lbm_set_geometry_host(h, _u8ptr(geo, n, "cpu"), int(wall_model)))


def lbm_boundary_force(h):
    F = np.empty(3)
    _check(load().lbm_boundary_force(h, F.ctypes.data))
    return F


def lbm_set_face_velocity(h, face, u=None):
    """u: float64 CUDA tensor [3*n] over the cells of the face (lower in-face axis fastest) or None (uniform face_u)."""
    _check(load().lbm_set_face_velocity(h, int(face), _ptr(u)))


def lbm_set_face_velocity_host(h, face, u=None):
    _check(load().lbm_set_face_velocity_host(h, int(face), _ptr(u, device="cpu")))


def lbm_set_face_density(h, rho6):
    r = np.ascontiguousarray(rho6, dtype=np.float64).reshape(6)
    _check(load().lbm_set_face_density(h, r.ctypes.data))


def lbm_init_equilibrium(h, rho=None, u=None):
    _check(load().lbm_init_equilibrium(h, _ptr(rho), _ptr(u)))


def lbm_init_equilibrium_host(h, rho=None, u=None):
    _check(load().lbm_init_equilibrium_host(h, _ptr(rho, device="cpu"), _ptr(u, device="cpu")))


def lbm_step(h, nsteps):
    _check(load().lbm_step(h, int(nsteps)))


def lbm_moments(h, rho=None, u=None, diagnostics=False):
    """Fills the given device tensors; returns the 8 diagnostics as a numpy array if asked."""
    diag = np.empty(8) if diagnostics else None
    _check(load().lbm_moments(h, _ptr(rho), _ptr(u), None if diag is None else diag.ctypes.data))
    return diag


def lbm_moments_host(h, rho=None, u=None, diagnostics=False):
    diag = np.empty(8) if diagnostics else None
    _check(load().lbm_moments_host(h, _ptr(rho, device="cpu"), _ptr(u, device="cpu"), None if diag is None else diag.ctypes.data))
    return diag


def lbm_diagnostics_static(f, lattice, out, force=None, stream=None):
    """The 8 diagnostics of `lbm_moments` for callers that may not allocate device memory and have no handle (a
    process whose GPU memory belongs to its own pool, a monitor inside a time loop that a cudaMalloc would stall,
    code that only holds a pointer to someone else's populations).  The library allocates nothing: its scratch is a
    fixed array inside the library, which is why grids beyond LBM_STATIC_MAX_CELLS cells are refused and why two
    calls that overlap on one GPU (different streams, no ordering) race.  See include/lbm.h.

    f: contiguous float64 CUDA tensor, Q*ncells canonical populations f[a*ncells + i]; lattice: Q, optionally
    | LBM_EQ_INCOMP; out: float64 CUDA tensor of 8 elements that receives the result (the caller passes it: this
    function creates no tensor); force: 3 floats or None; stream: raw cudaStream_t (int) or None = default stream.
    Asynchronous: read `out` after synchronising the stream."""
    Q = int(lattice) & 0xFF
    assert Q > 0 and f.numel() % Q == 0, (f.numel(), Q)
    fo = None if force is None else np.ascontiguousarray(force, dtype=np.float64).reshape(3)
    _check(load().lbm_diagnostics_static(_ptr(f), f.numel() // Q, int(lattice), None if fo is None else fo.ctypes.data,
                                         _ptr(out, 8), None if stream is None else int(stream)))


def lbm_get_populations(h, f):
    _check(load().lbm_get_populations(h, _ptr(f)))


def lbm_set_populations(h, f):
    _check(load().lbm_set_populations(h, _ptr(f)))


def lbm_lattice(lattice):
    Q = lattice & 0xFF
    e = (C.c_int32 * (3 * Q))()
    t = (C.c_double * Q)()
    _check(load().lbm_lattice(int(lattice), e, t))
    return np.array(e, dtype=np.int32).reshape(Q, 3), np.array(t, dtype=np.float64)


def lbm_time(h) -> int:
    return int(load().lbm_time(h))


def lbm_launch_count(h) -> int:
    return int(load().lbm_launch_count(h))


def lbm_set_block(h, bx, by):
    _check(load().lbm_set_block(h, int(bx), int(by)))


def lbm_debug_arm(h, poison=True):
    _check(load().lbm_debug_arm(h, 1 if poison else 0))


def lbm_debug_check(h) -> int:
    n = int(load().lbm_debug_check(h))
    if n < 0:
        raise LBMError(n, lbm_last_error())
    return n


def lbm_set_persistent(h, on):
    _check(load().lbm_set_persistent(h, 1 if on else 0))


def lbm_set_two_step(h, on):
    """0: never; 1 (default): where it pays; 2: wherever stream_collide_ab2 exists."""
    _check(load().lbm_set_two_step(h, int(on)))


# ---- convenience wrapper ----------------------------------------------------------------
class Solver:
    """Owns one handle.  All tensors are torch float64, on the solver's CUDA device unless the
    method name says host."""

    def __init__(self, nx, ny, nz, Q=19, tau=0.8, eq=LBM_EQ_STANDARD, scheme=LBM_SCHEME_AUTO, store=LBM_STORE_F64,
                 face_kind=None, face_u=None, force=None, stream=None, layout=LBM_LAYOUT_ROWS):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2201_11330_b200 needs a CUDA device (no CPU fallback)")
        self.nx, self.ny, self.nz, self.Q = int(nx), int(ny), int(nz), int(Q)
        self.N = self.nx * self.ny * self.nz
        self.torch_stream = stream  # torch.cuda.Stream or None
        raw = None if stream is None else stream.cuda_stream
        self.bc = make_bc(face_kind, face_u, force, raw)
        self.h = lbm_create(nx, ny, nz, int(Q) | eq | scheme | store | layout, tau, self.bc)

    @classmethod
    def from_workload(cls, w, **kw):
        """Solver for an inputs.Workload, geometry (solid mask, wall model) included."""
        import torch
        eq = LBM_EQ_INCOMP if getattr(w, "eq", 0) else LBM_EQ_STANDARD
        s = cls(w.nx, w.ny, w.nz, w.Q, w.tau, eq=eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force, **kw)
        if getattr(w, "has_geometry", False):
            geo = w.geo()
            s.set_geometry(None if geo is None else torch.from_numpy(geo), w.wall_model)
        if getattr(w, "face_rho", None) is not None:
            s.set_face_density(w.face_rho)
        for face, prof in getattr(w, "face_profiles", dict)().items():
            s.set_face_velocity(face, torch.from_numpy(np.ascontiguousarray(prof).reshape(-1)))
        return s

    def close(self):
        if getattr(self, "h", None):
            lbm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_geometry(self, geo=None, wall_model=LBM_WALL_HALFWAY):
        """geo: uint8 tensor of N bytes (CUDA or CPU; non-zero = solid) or None."""
        if geo is not None and geo.device.type == "cpu":
            lbm_set_geometry_host(self.h, geo, wall_model, self.N)
        else:
            lbm_set_geometry(self.h, geo, wall_model, self.N)

    def boundary_force(self):
        return lbm_boundary_force(self.h)

    def set_face_velocity(self, face, u=None):
        """Per-cell wall velocity of MOVING face `face`: float64 tensor [3*n] (CUDA or CPU) or None."""
        if u is not None and u.device.type == "cpu":
            lbm_set_face_velocity_host(self.h, face, u)
        else:
            lbm_set_face_velocity(self.h, face, u)

    def set_face_density(self, rho6):
        lbm_set_face_density(self.h, rho6)

    def init_equilibrium(self, rho=None, u=None):
        self._before()
        lbm_init_equilibrium(self.h, rho, u)
        self._after(rho, u)

    def init_equilibrium_host(self, rho=None, u=None):
        # Contract (include/lbm.h): the library returns once rho / u have left the host, so temporaries such as
        # `x.pin_memory()` passed inline may be dropped by the caller right away — torch's pinned-memory cache can
        # recycle their blocks without racing the library's internal copy stream.  No reference is kept here.
        lbm_init_equilibrium_host(self.h, rho, u)

    def step(self, n=1):
        lbm_step(self.h, n)

    # The library works on the handle's stream; tensors handed over or returned here belong to torch's current stream.
    # _before / _after order the two (no-ops when they are the same stream) so that a temporary is not recycled while a
    # kernel still reads it and a result is not read before it has been written.
    def _before(self):
        import torch
        cur = torch.cuda.current_stream()
        if self.torch_stream is not None:
            self.torch_stream.wait_stream(cur)
        elif cur != torch.cuda.default_stream():
            cur.synchronize()  # the handle runs on the default stream, torch on another one

    def _after(self, *tensors):
        import torch
        cur = torch.cuda.current_stream()
        if self.torch_stream is not None:
            cur.wait_stream(self.torch_stream)
            for t in tensors:
                if t is not None:
                    t.record_stream(self.torch_stream)
        elif cur != torch.cuda.default_stream():
            torch.cuda.default_stream().synchronize()

    def moments(self, fields=True, diagnostics=True):
        import torch
        rho = torch.empty(self.N, dtype=torch.float64, device="cuda") if fields else None
        u = torch.empty(3 * self.N, dtype=torch.float64, device="cuda") if fields else None
        self._before()
        diag = lbm_moments(self.h, rho, u, diagnostics)
        self._after(rho, u)
        return rho, (None if u is None else u.view(3, self.N)), diag

    def diagnostics(self):
        return lbm_moments(self.h, None, None, True)

    def get_populations(self, out=None):
        import torch
        f = torch.empty(self.Q * self.N, dtype=torch.float64, device="cuda") if out is None else out
        self._before()
        lbm_get_populations(self.h, f)
        self._after(f)
        return f.view(self.Q, self.N)

    def set_populations(self, f):
        f = f.contiguous().view(-1)
        self._before()
        lbm_set_populations(self.h, f)
        self._after(f)

    @property
    def time(self):
        return lbm_time(self.h)

    @property
    def launches(self):
        return lbm_launch_count(self.h)

    def set_block(self, bx, by):
        lbm_set_block(self.h, bx, by)

    def set_persistent(self, on):
        lbm_set_persistent(self.h, on)

    def set_two_step(self, on):
        lbm_set_two_step(self.h, on)

    def debug_arm(self, poison=True):
        lbm_debug_arm(self.h, poison)

    def debug_check(self) -> int:
        return lbm_debug_check(self.h)
