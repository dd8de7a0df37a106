"""z-slab decomposition of one box over several GPUs (include/lbm.h "z-slab decomposition"; R21, §8).

The paper splits the box into Cartesian MPI blocks, one per device, and exchanges the populations that
cross a cut once per step through host-staged MPI.  Here the cut is along
z only, the exchange is done by the fused step kernel itself (peer stores into the neighbour's halo plane)
and the ordering between slabs is a device-side step counter; this module is the host-side plumbing:

  partition / neighbours / halo_box / slab_mask / combine_diagnostics   pure functions (tested on CPU)
  exchange_descriptors, all_reduce_diagnostics               torch.distributed (gloo on CPU, nccl on GPUs)
  SlabSolver                                                 one slab = one rank's share (one process per GPU)
  SlabGroup                                                  all slabs of a box in ONE process (one or more devices)

No lattice-Boltzmann arithmetic happens here.
"""
from __future__ import annotations

import numpy as np

from . import lbm


# ------------------------------------------------------------------------------------------ pure host logic
def partition(nz: int, world: int):
    """Balanced split of nz planes into `world` slabs of whole planes: [(z0, nz_local)], larger slabs first."""
    if world < 1 or nz < world:
        raise ValueError(f"cannot cut {nz} planes into {world} slabs of at least one plane")
    base, extra = divmod(nz, world)
    out, z0 = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((z0, n))
        z0 += n
    return out


def neighbours(rank: int, world: int, periodic_z: bool):
    """(lower, upper) rank of a slab, None where the box ends at a non-periodic z face.  A periodic box of one
    slab is its own neighbour on both sides."""
    lower = rank - 1 if rank > 0 else (world - 1 if periodic_z else None)
    upper = rank + 1 if rank < world - 1 else (0 if periodic_z else None)
    return lower, upper


def halo_box(nx: int, ny: int, z0: int, nz_local: int):
    """Sub-box of the global grid that a slab's arrays cover: its own planes plus one halo plane on each side
    (inputs.Workload.fields(box=...) wraps the coordinates periodically)."""
    return ((0, nx), (0, ny), (z0 - 1, z0 + nz_local + 1))


def slab_mask(geo, nx: int, ny: int, nz: int, z0: int, nz_local: int, periodic_z: bool):
    """The solid mask a slab hands to lbm_set_geometry: its own planes plus TWO halo planes per side
    (include/lbm.h: the wall-node status of a halo node depends on the plane beyond it), uint8[(nz_local+4)*ny*nx].
    geo: uint8[nz*ny*nx] of the whole box or None.  Periodic z wraps; beyond a non-periodic z face the planes are 0."""
    out = np.zeros((nz_local + 4, ny * nx), dtype=np.uint8)
    if geo is None:
        return out.reshape(-1)
    g = np.asarray(geo, dtype=np.uint8).reshape(nz, ny * nx)
    for k in range(nz_local + 4):
        z = z0 - 2 + k
        if periodic_z:
            out[k] = g[z % nz]
        elif 0 <= z < nz:
            out[k] = g[z]
    return out.reshape(-1)


def combine_diagnostics(parts):
    """The 8 diagnostics of the whole box from those of its slabs: sums, max |u|, min rho, non-finite count."""
    parts = np.asarray(list(parts), dtype=np.float64).reshape(-1, 8)
    out = parts.sum(axis=0)
    out[5] = parts[:, 5].max()
    out[6] = parts[:, 6].min()
    return out


def strip_halo(a, nx: int, ny: int, nz_local: int, comps: int = 1):
    """Own planes of a slab array laid out [comps][nz_local+2][ny][nx] -> [comps][nz_local*ny*nx]."""
    v = a.reshape(comps, nz_local + 2, ny * nx)[:, 1:-1, :]
    return v.reshape(comps, nz_local * ny * nx)


# ------------------------------------------------------------------------------------------ torch.distributed
def exchange_descriptors(desc_bytes: bytes):
    """All ranks' slab descriptors (bytes of lbm_slab_peer_t), in rank order."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return [desc_bytes]
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, desc_bytes)
    return out


def all_reduce_diagnostics(diag, device="cpu"):
    """combine_diagnostics across the ranks of the process group (three small all-reduces: SUM, MAX, MIN)."""
    import torch
    import torch.distributed as dist
    d = np.asarray(diag, dtype=np.float64).copy()
    if not (dist.is_available() and dist.is_initialized()):
        return d
    sums = torch.tensor(d, dtype=torch.float64, device=device)
    mx = torch.tensor([d[5]], dtype=torch.float64, device=device)
    mn = torch.tensor([d[6]], dtype=torch.float64, device=device)
    dist.all_reduce(sums, op=dist.ReduceOp.SUM)
    dist.all_reduce(mx, op=dist.ReduceOp.MAX)
    dist.all_reduce(mn, op=dist.ReduceOp.MIN)
    out = sums.cpu().numpy()
    out[5] = float(mx.item())
    out[6] = float(mn.item())
    return out


def _peer_from_bytes(b: bytes) -> lbm.lbm_slab_peer_t:
    return lbm.lbm_slab_peer_t.from_buffer_copy(b)


# ------------------------------------------------------------------------------------------ one slab
class Slab:
    """One z-slab handle with its placement; arrays at its interface cover nz_local + 2 planes."""

    def __init__(self, w, z0, nz_local, scheme=lbm.LBM_SCHEME_AB, store=lbm.LBM_STORE_F64, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2201_11330_b200 needs a CUDA device (no CPU fallback)")
        self.w, self.z0, self.nz_local = w, int(z0), int(nz_local)
        self.nx, self.ny, self.Q = w.nx, w.ny, w.Q
        self.N = self.nx * self.ny * (self.nz_local + 2)
        self.N_own = self.nx * self.ny * self.nz_local
        self.device = torch.cuda.current_device()
        self.torch_stream = stream
        eq = lbm.LBM_EQ_INCOMP if getattr(w, "eq", 0) else lbm.LBM_EQ_STANDARD
        self.bc = lbm.make_bc(w.face_kind, w.face_u, w.force, None if stream is None else stream.cuda_stream)
        self.h = lbm.lbm_create_slab(self.nx, self.ny, self.nz_local, self.z0, w.nz, int(w.Q) | eq | scheme | store, w.tau, self.bc)
        # solid mask and wall model: the slab's planes of the whole-box mask + two halo planes per side
        self.has_geometry = bool(getattr(w, "has_geometry", False))
        if self.has_geometry:
            m = slab_mask(w.geo(), self.nx, self.ny, w.nz, self.z0, self.nz_local, w.face_kind[4] == 0)
            lbm.lbm_set_geometry(self.h, torch.from_numpy(m).cuda(), w.wall_model, m.size)
        # open boundaries (D:R22): every slab takes the density and the per-cell velocity of the WHOLE box faces
        if getattr(w, "face_rho", None) is not None:
            lbm.lbm_set_face_density(self.h, w.face_rho)
        for face, prof in getattr(w, "face_profiles", dict)().items():
            lbm.lbm_set_face_velocity(self.h, face, torch.from_numpy(np.ascontiguousarray(prof).reshape(-1)).cuda())

    def descriptor(self) -> bytes:
        return bytes(lbm.lbm_slab_export(self.h))

    def connect(self, lower: bytes | None, upper: bytes | None):
        lbm.lbm_slab_connect(self.h, None if lower is None else _peer_from_bytes(lower),
                             None if upper is None else _peer_from_bytes(upper))

    def fields(self):
        """(rho, u) of the workload on this slab's planes + halo planes (numpy; seeded, point-wise recipe)."""
        return self.w.fields(box=halo_box(self.nx, self.ny, self.z0, self.nz_local))

    def init_equilibrium(self, rho=None, u=None):
        """rho[N], u[3N] device tensors WITH halo planes; default: the workload's own fields."""
        import torch
        if rho is None and u is None:
            r, v = self.fields()
            rho = torch.from_numpy(r).cuda()
            u = torch.from_numpy(np.ascontiguousarray(v.reshape(-1))).cuda()
        lbm.lbm_init_equilibrium(self.h, rho, u)

    def step(self, n=1):
        lbm.lbm_step(self.h, n)

    def diagnostics(self):
        return lbm.lbm_moments(self.h, None, None, True)

    def boundary_force(self):
        """This slab's part of the momentum-exchange force (Eq. 13): the links of its own fluid nodes."""
        return lbm.lbm_boundary_force(self.h)

    def moments(self):
        """(rho[N_own], u[3, N_own]) of the own planes (device tensors), diagnostics of the own planes."""
        import torch
        rho = torch.zeros(self.N, dtype=torch.float64, device="cuda")
        u = torch.zeros(3 * self.N, dtype=torch.float64, device="cuda")
        d = lbm.lbm_moments(self.h, rho, u, True)
        return (strip_halo(rho, self.nx, self.ny, self.nz_local)[0], strip_halo(u, self.nx, self.ny, self.nz_local, 3), d)

    def get_populations(self):
        """Canonical populations of the own planes, [Q, N_own] (device tensor)."""
        import torch
        f = torch.zeros(self.Q * self.N, dtype=torch.float64, device="cuda")
        lbm.lbm_get_populations(self.h, f)
        return strip_halo(f, self.nx, self.ny, self.nz_local, self.Q)

    def set_populations(self, f_with_halo):
        lbm.lbm_set_populations(self.h, f_with_halo.contiguous().view(-1))

    @property
    def launches(self):
        return lbm.lbm_launch_count(self.h)

    def close(self):
        if getattr(self, "h", None):
            lbm.lbm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class SlabSolver(Slab):
    """This rank's slab of workload w under torch.distributed (one process per GPU): creates the slab, exchanges
    the descriptors, connects to the neighbours' memory (CUDA IPC -> NVLink peer stores)."""

    def __init__(self, w, rank, world, device_sync=True, **kw):
        self.rank, self.world = rank, world
        z0, nzl = partition(w.nz, world)[rank]
        super().__init__(w, z0, nzl, **kw)
        descs = exchange_descriptors(self.descriptor())
        lo, up = neighbours(rank, world, w.face_kind[4] == 0)
        self.connect(None if lo is None else descs[lo], None if up is None else descs[up])
        if not device_sync:
            lbm.lbm_slab_set_sync(self.h, False)

    def global_diagnostics(self, device="cuda"):
        return all_reduce_diagnostics(self.diagnostics(), device)

    def global_boundary_force(self, device="cuda"):
        """Eq. 13 of the whole box: the slabs' parts summed over the process group."""
        import torch
        import torch.distributed as dist
        F = torch.tensor(self.boundary_force(), dtype=torch.float64, device=device)
        if dist.is_available() and dist.is_initialized():
            dist.all_reduce(F, op=dist.ReduceOp.SUM)
        return F.cpu().numpy()


class SlabGroup:
    """All slabs of a box in one process: slab r on devices[r % len(devices)], each on its own stream.
    Used to test the slab path on one GPU and to drive several GPUs from one process.
    shared_stream=True: every slab on the default stream instead, host-ordered (lbm_slab_set_sync(h, 0) before the
    connect, include/lbm.h): step() issues one step per slab in turn and the one stream keeps them in order."""

    def __init__(self, w, nslabs, devices=None, shared_stream=False, **kw):
        import torch
        self.w = w
        self.devices = list(devices) if devices else [torch.cuda.current_device()]
        self.slabs = []
        self.parts = partition(w.nz, nslabs)
        for r, (z0, nzl) in enumerate(self.parts):
            with torch.cuda.device(self._dev(r)):
                self.slabs.append(Slab(w, z0, nzl, stream=None if shared_stream else torch.cuda.Stream(), **kw))
                if shared_stream:
                    lbm.lbm_slab_set_sync(self.slabs[-1].h, False)
        descs = [s.descriptor() for s in self.slabs]
        for r, s in enumerate(self.slabs):
            lo, up = neighbours(r, nslabs, w.face_kind[4] == 0)
            with torch.cuda.device(self._dev(r)):
                s.connect(None if lo is None else descs[lo], None if up is None else descs[up])

    def _dev(self, r):
        return self.devices[r % len(self.devices)]

    def _each(self, fn):
        import torch
        out = []
        for r, s in enumerate(self.slabs):
            with torch.cuda.device(self._dev(r)), torch.cuda.stream(s.torch_stream):
                out.append(fn(s))
        return out

    def synchronize(self):
        import torch
        for r, s in enumerate(self.slabs):
            if s.torch_stream is not None:
                s.torch_stream.synchronize()
            else:
                torch.cuda.default_stream(self._dev(r)).synchronize()

    def init_equilibrium(self):
        self.synchronize()
        self._each(lambda s: s.init_equilibrium())
        self.synchronize()

    def step(self, n=1):
        # one step per slab in turn: no stream ever queues far ahead of the neighbours it waits for
        for _ in range(n):
            for s in self.slabs:
                s.step(1)

    def diagnostics(self):
        return combine_diagnostics(self._each(lambda s: s.diagnostics()))

    def boundary_force(self):
        return np.sum(self._each(lambda s: s.boundary_force()), axis=0)

    def get_populations(self):
        """Canonical populations of the whole box, [Q, N] (on the first device)."""
        import torch
        parts = self._each(lambda s: s.get_populations().view(s.Q, s.nz_local, -1))
        self.synchronize()
        dev = parts[0].device
        return torch.cat([p.to(dev) for p in parts], dim=1).reshape(self.w.Q, -1)

    def moments(self):
        import torch
        parts = self._each(lambda s: s.moments())
        self.synchronize()
        dev = parts[0][0].device
        rho = torch.cat([p[0].to(dev) for p in parts])
        u = torch.cat([p[1].view(3, s.nz_local, -1).to(dev) for p, s in zip(parts, self.slabs)], dim=1).reshape(3, -1)
        return rho, u, combine_diagnostics([p[2] for p in parts])

    @property
    def launches(self):
        return sum(s.launches for s in self.slabs)

    def close(self):
        self.synchronize()
        for s in self.slabs:
            s.close()
