"""CPU tests of the host-side logic of the z-slab decomposition (paper_2201_11330_b200/slabs.py): the partition,
the neighbour map, the halo boxes of the seeded inputs, the combination of the per-slab diagnostics, and — with
two gloo processes — the exchange of slab descriptors and the three all-reduces of the diagnostics."""
import json
import re
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2201_11330_b200 import inputs, lbm, slabs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("nz,world", [(512, 8), (512, 3), (7, 7), (13, 4), (5, 1)])
def test_partition_covers_every_plane_once(nz, world):
    parts = slabs.partition(nz, world)
    assert len(parts) == world and parts[0][0] == 0
    assert all(n >= 1 for _, n in parts)
    assert max(n for _, n in parts) - min(n for _, n in parts) <= 1
    covered = [z for z0, n in parts for z in range(z0, z0 + n)]
    assert covered == list(range(nz))


def test_partition_refuses_more_slabs_than_planes():
    with pytest.raises(ValueError):
        slabs.partition(3, 4)
    with pytest.raises(ValueError):
        slabs.partition(3, 0)


def test_neighbours():
    assert slabs.neighbours(0, 4, True) == (3, 1)
    assert slabs.neighbours(3, 4, True) == (2, 0)
    assert slabs.neighbours(0, 4, False) == (None, 1)
    assert slabs.neighbours(3, 4, False) == (2, None)
    assert slabs.neighbours(0, 1, True) == (0, 0)  # a periodic box of one slab is its own neighbour
    assert slabs.neighbours(0, 1, False) == (None, None)
    # symmetric: if a is b's upper neighbour, b is a's lower one
    for world in (2, 3, 5):
        for per in (True, False):
            for r in range(world):
                lo, up = slabs.neighbours(r, world, per)
                if up is not None:
                    assert slabs.neighbours(up, world, per)[0] == r
                if lo is not None:
                    assert slabs.neighbours(lo, world, per)[1] == r


def test_halo_fields_are_slices_of_the_global_fields():
    """The point-wise input recipe on a slab's halo box equals the global field's planes, periodic wrap included."""
    w = inputs.Workload("t", 6, 5, 9, 19, 0.8, 1, u0=0.05, noise=1e-3, seed=inputs.SEED_BASE + 3)
    rho, u = w.fields()
    rho = rho.reshape(w.nz, -1)
    u = u.reshape(3, w.nz, -1)
    for z0, nzl in slabs.partition(w.nz, 4):
        r, v = w.fields(box=slabs.halo_box(w.nx, w.ny, z0, nzl))
        zs = [(z0 - 1 + k) % w.nz for k in range(nzl + 2)]
        assert np.array_equal(r.reshape(nzl + 2, -1), rho[zs])
        assert np.array_equal(v.reshape(3, nzl + 2, -1), u[:, zs])
        own = slabs.strip_halo(r, w.nx, w.ny, nzl)
        assert np.array_equal(own[0], rho[z0:z0 + nzl].reshape(-1))


def test_combine_diagnostics():
    a = np.array([10.0, 1.0, 2.0, 3.0, 0.5, 0.07, 0.99, 0.0])
    b = np.array([20.0, -1.0, 0.5, 1.0, 0.25, 0.09, 0.98, 2.0])
    c = slabs.combine_diagnostics([a, b])
    assert c.tolist() == [30.0, 0.0, 2.5, 4.0, 0.75, 0.09, 0.98, 2.0]
    assert slabs.combine_diagnostics([a]).tolist() == a.tolist()


def test_descriptor_struct_matches_the_header():
    """lbm_slab_peer_t in the binding has the size and field order of include/lbm.h (plain bytes cross processes)."""
    import ctypes as C
    # buf[2], flags, plane_stride | nz_local, device | pid | Q, elem_bytes, layout_soa, reserved | stream | ipc handles
    assert C.sizeof(lbm.lbm_slab_peer_t) == 2 * 8 + 8 + 8 + 4 + 4 + 8 + 4 * 4 + 8 + 2 * 64 + 64
    d = lbm.lbm_slab_peer_t()
    d.buf[0], d.buf[1], d.flags, d.plane_stride, d.nz_local, d.device, d.pid = 1, 2, 3, 4, 5, 6, 7
    back = lbm.lbm_slab_peer_t.from_buffer_copy(bytes(d))
    assert (back.buf[0], back.buf[1], back.flags, back.plane_stride, back.nz_local, back.device, back.pid) == (1, 2, 3, 4, 5, 6, 7)
    src = open(os.path.join(ROOT, "include", "lbm.h")).read()
    body = src[src.index("typedef struct {\n  uint64_t buf[2];"):src.index("} lbm_slab_peer_t;")]
    order = [ln.split(";")[0].split()[-1].split("[")[0] for ln in body.splitlines()[1:] if ";" in ln]
    assert order == [n for n, _ in lbm.lbm_slab_peer_t._fields_]


WORKER = r"""
import os, sys, json
import numpy as np
sys.path.insert(0, os.environ["LBM_ROOT"])
from paper_2201_11330_b200 import replicas, slabs, lbm
rank, local_rank, world = replicas.init(backend="gloo")
assert world == 2
z0, nzl = slabs.partition(9, world)[rank]
d = lbm.lbm_slab_peer_t()
d.buf[0], d.nz_local, d.pid, d.plane_stride = 1000 + rank, nzl, os.getpid(), 6 * 5 * (nzl + 2)
descs = slabs.exchange_descriptors(bytes(d))
got = [lbm.lbm_slab_peer_t.from_buffer_copy(b) for b in descs]
lo, up = slabs.neighbours(rank, world, True)
diag = np.array([10.0 * (rank + 1), rank, -rank, 1.0, 0.5, 0.01 * (rank + 1), 1.0 - 0.1 * rank, rank], dtype=np.float64)
tot = slabs.all_reduce_diagnostics(diag)
replicas.barrier()
print("OUT" + json.dumps({"rank": rank, "bufs": [int(g.buf[0]) for g in got], "nzl": [int(g.nz_local) for g in got],
                          "pids_differ": got[0].pid != got[1].pid, "lo": lo, "up": up, "tot": tot.tolist()}), flush=True)
replicas.finalize()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_descriptor_exchange_and_diagnostics_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, LBM_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    # the two ranks share one pipe: their lines can arrive glued together
    outs = [json.loads(m) for m in re.findall(r"OUT(\{[^{}]*\})", r.stdout)]
    assert len(outs) == 2
    for o in outs:
        assert o["bufs"] == [1000, 1001] and o["nzl"] == [5, 4] and o["pids_differ"]
        assert (o["lo"], o["up"]) == ((1, 1) if o["rank"] == 0 else (0, 0))
        assert o["tot"] == [30.0, 1.0, -1.0, 2.0, 1.0, 0.02, 0.9, 1.0]


def test_slab_mask_carries_two_halo_planes_per_side():
    """include/lbm.h: on a slab lbm_set_geometry takes nz_local + 4 planes, plane 2 + (z - z0); periodic z wraps, planes
    beyond a non-periodic z face are empty."""
    nx, ny, nz = 4, 3, 7
    geo = (np.arange(nx * ny * nz) % 3 == 0).astype(np.uint8)
    g = geo.reshape(nz, ny * nx)
    for z0, nzl in slabs.partition(nz, 3):
        m = slabs.slab_mask(geo, nx, ny, nz, z0, nzl, True).reshape(nzl + 4, ny * nx)
        for k in range(nzl + 4):
            assert (m[k] == g[(z0 - 2 + k) % nz]).all()
        m = slabs.slab_mask(geo, nx, ny, nz, z0, nzl, False).reshape(nzl + 4, ny * nx)
        for k in range(nzl + 4):
            z = z0 - 2 + k
            assert (m[k] == (g[z] if 0 <= z < nz else 0)).all()
    assert slabs.slab_mask(None, nx, ny, nz, 0, 3, True).sum() == 0
