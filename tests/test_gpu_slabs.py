"""GPU parity of the z-slab decomposition (include/lbm.h "z-slab decomposition", R21): a box cut into
slabs whose fused step kernels fill each other's halo planes must give, cell for cell, the populations of the
undivided box — bit for bit against the single-handle CUDA run (same arithmetic per cell), and within 1e-12 of
the CPU oracle.  All slabs live on ONE device here (separate streams, device-side step counters); nothing in
these tests makes a kernel wait for another kernel.
"""
import numpy as np
import pytest

from oracle import Oracle
from oracle.binding import EQ_INCOMP, EQ_STANDARD
from paper_2201_11330_b200 import inputs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
TOL = 1e-12
B, M, P = inputs.FACE_BOUNCE, inputs.FACE_MOVING, inputs.FACE_PERIODIC


@pytest.fixture(scope="module")
def mods():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_11330_b200 import lbm, slabs
    lbm.load()
    return lbm, slabs


def workload(dims, Q, tau, faces=None, face_u=None, force=(0.0, 0.0, 0.0), eq=EQ_STANDARD, kind="tgv", steps=8):
    fu = np.zeros((6, 3))
    for k, v in (face_u or {}).items():
        fu[k] = v
    return inputs.Workload(f"slabtest_{Q}_{dims}", dims[0], dims[1], dims[2], Q, tau, steps,
                           face_kind=tuple(faces or [P] * 6), face_u=tuple(map(tuple, fu)), force=tuple(force),
                           u0=0.05, noise=1e-3, seed=inputs.SEED_BASE + 77, kind=kind, eq=eq)


def oracle_run(w, steps):
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force)
    o.init_equilibrium(rho, u)
    o.step(steps)
    f = o.get_f()
    d = o.moments(False)[2]
    o.close()
    return f, d


def single_run(lbm, w, steps, store=0):
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w, scheme=lbm.LBM_SCHEME_AB, store=store)
    s.init_equilibrium(torch.from_numpy(rho).cuda(), torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda())
    s.step(steps)
    f = s.get_populations().clone()
    d = s.diagnostics()
    s.close()
    return f, d


CASES = {
    "tgv_periodic_q19": dict(dims=(24, 20, 22), Q=19, tau=0.8),
    "channel_zwalls_q27_forced": dict(dims=(20, 12, 13), Q=27, tau=0.9, faces=[P, P, P, P, B, B], force=(1e-5, 2e-6, 0.0), kind="rest"),
    "cavity_lid_q19": dict(dims=(16, 14, 12), Q=19, tau=0.55, faces=[B, B, B, B, B, M], face_u={5: (0.1, 0.0, 0.0)}, kind="rest"),
    "moving_zlo_and_x_q27": dict(dims=(12, 10, 9), Q=27, tau=0.7, faces=[B, M, P, P, M, B],
                                 face_u={1: (0.0, 0.03, -0.02), 4: (0.05, 0.01, 0.0)}, kind="rest"),
    "incomp_forced_q19": dict(dims=(40, 6, 10), Q=19, tau=0.62, eq=EQ_INCOMP, force=(0.0, 1e-5, -3e-6)),
    "d2q9_planes": dict(dims=(33, 17, 5), Q=9, tau=0.7),
}


@pytest.mark.parametrize("nslabs", [1, 2, 3])
@pytest.mark.parametrize("case", list(CASES))
def test_slabs_equal_the_undivided_box(mods, case, nslabs):
    lbm, slabs = mods
    w = workload(**CASES[case])
    ref, dref = oracle_run(w, w.steps)
    one, d1 = single_run(lbm, w, w.steps)
    g = slabs.SlabGroup(w, nslabs)
    g.init_equilibrium()
    g.step(w.steps)
    f = g.get_populations()
    d = g.diagnostics()
    launches = g.launches
    g.close()
    assert launches >= nslabs * w.steps
    assert torch.equal(f, one), f"{case}: slabs differ from the undivided CUDA run by {float((f - one).abs().max())}"
    assert float(np.abs(f.cpu().numpy() - ref).max()) <= TOL
    # sums are order dependent (R14): relative 1e-12; max / min exact
    for k in (0, 4):
        assert abs(d[k] - dref[k]) <= 1e-12 * max(1.0, abs(dref[k]))
    assert d[5] == d1[5] and d[6] == d1[6] and d[7] == 0


def test_one_plane_slabs_and_ragged_split(mods):
    """nz = 7 cut into 7 slabs of one plane (both pushes come from the same plane) and into 4 ragged slabs."""
    lbm, slabs = mods
    w = workload((18, 9, 7), 19, 0.6, steps=10)
    one, _ = single_run(lbm, w, w.steps)
    for n in (7, 4):
        g = slabs.SlabGroup(w, n)
        assert [p[1] for p in g.parts] == ([1] * 7 if n == 7 else [2, 2, 2, 1])
        g.init_equilibrium()
        g.step(w.steps)
        f = g.get_populations()
        g.close()
        assert torch.equal(f, one)


def test_random_populations_through_set_populations(mods):
    """Non-equilibrium state handed over WITH halo planes (the interface contract of a slab)."""
    lbm, slabs = mods
    w = workload((10, 12, 9), 27, 0.75, faces=[P, P, B, B, P, P], kind="rest")
    rng = np.random.default_rng(5)
    f0 = (1.0 / 27) * (1.0 + 0.2 * rng.uniform(-1, 1, (27, w.nz, w.ny * w.nx)))
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, face_kind=w.face_kind)
    o.set_f(f0.reshape(27, -1))
    o.step(5)
    ref = o.get_f()
    o.close()
    g = slabs.SlabGroup(w, 3)
    for s in g.slabs:
        zs = [(s.z0 - 1 + k) % w.nz for k in range(s.nz_local + 2)]
        s.set_populations(torch.from_numpy(np.ascontiguousarray(f0[:, zs, :])).cuda())
    torch.cuda.synchronize()
    g.step(5)
    f = g.get_populations()
    g.close()
    assert float(np.abs(f.cpu().numpy() - ref).max()) <= TOL


def test_fp32_storage_slabs_equal_the_undivided_fp32_run(mods):
    lbm, slabs = mods
    w = workload((32, 8, 12), 19, 0.8, steps=12)
    one, _ = single_run(lbm, w, w.steps, store=lbm.LBM_STORE_F32)
    g = slabs.SlabGroup(w, 3, store=lbm.LBM_STORE_F32)
    g.init_equilibrium()
    g.step(w.steps)
    f = g.get_populations()
    g.close()
    assert torch.equal(f, one)


def test_host_synchronised_mode(mods):
    """lbm_slab_set_sync(0): no device-side counters, the caller synchronises all slabs between steps."""
    lbm, slabs = mods
    w = workload((16, 8, 10), 19, 0.7, steps=6)
    one, _ = single_run(lbm, w, w.steps)
    g = slabs.SlabGroup(w, 2)
    for s in g.slabs:
        lbm.lbm_slab_set_sync(s.h, False)
    g.init_equilibrium()
    for _ in range(w.steps):
        g.step(1)
        g.synchronize()
    f = g.get_populations()
    g.close()
    assert torch.equal(f, one)


def test_host_ordered_slabs_may_share_a_stream(mods):
    """Device-side ordering needs a stream per slab (a step would wait for one queued behind it) and lbm_slab_connect
    refuses a shared one; host-ordered slabs (lbm_slab_set_sync(h, 0) BEFORE the connect) may all sit on the default
    stream, which then orders the steps issued slab by slab — no synchronisation between steps at all."""
    lbm, slabs = mods
    w = workload((16, 8, 10), 19, 0.7, steps=6)
    one, _ = single_run(lbm, w, w.steps)
    a, b = slabs.Slab(w, 0, 5), slabs.Slab(w, 5, 5)  # both on the default stream, device-side ordering still on
    with pytest.raises(lbm.LBMError) as ei:
        a.connect(b.descriptor(), b.descriptor())
    assert ei.value.code == lbm.LBM_EINVAL and "lbm_slab_set_sync" in str(ei.value)
    a.close()
    b.close()
    g = slabs.SlabGroup(w, 3, shared_stream=True)
    with pytest.raises(lbm.LBMError):
        lbm.lbm_slab_set_sync(g.slabs[0].h, True)  # would deadlock on the shared stream
    g.init_equilibrium()
    g.step(w.steps)
    f = g.get_populations()
    g.close()
    assert torch.equal(f, one)


def test_moments_fields_of_the_slabs(mods):
    lbm, slabs = mods
    w = workload((12, 10, 8), 19, 0.9, faces=[P, P, P, P, B, B], force=(2e-5, 0.0, 0.0), kind="rest", steps=7)
    rho0, u0 = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, face_kind=w.face_kind, force=w.force)
    o.init_equilibrium(rho0, u0)
    o.step(w.steps)
    rr, ur, dr = o.moments(True)
    o.close()
    g = slabs.SlabGroup(w, 3)
    g.init_equilibrium()
    g.step(w.steps)
    rho, u, d = g.moments()
    g.close()
    assert float(np.abs(rho.cpu().numpy() - rr).max()) <= 1e-13
    assert float(np.abs(u.cpu().numpy() - ur.reshape(3, -1)).max()) <= 1e-13
    assert abs(d[1] - dr[1]) <= 1e-12 * max(1.0, abs(dr[1]))


def test_slab_argument_errors(mods):
    lbm, slabs = mods
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create_slab(8, 8, 4, 6, 8, 19, 0.8)  # z0 + nz_local > nz_global
    with pytest.raises(lbm.LBMError):
        lbm.lbm_create_slab(8, 8, 0, 0, 8, 19, 0.8)
    with pytest.raises(lbm.LBMError) as ei:
        lbm.lbm_create_slab(8, 8, 4, 0, 8, 19 | lbm.LBM_SCHEME_AA, 0.8)
    assert ei.value.code == lbm.LBM_EINVAL or "LBM_SCHEME_AB" in str(ei.value)
    h = lbm.lbm_create_slab(8, 8, 4, 0, 8, 19, 0.8)
    other = lbm.lbm_create_slab(6, 8, 4, 4, 8, 19, 0.8)  # different nx
    try:
        with pytest.raises(lbm.LBMError):
            lbm.lbm_slab_connect(h, lbm.lbm_slab_export(other), None)
        with pytest.raises(lbm.LBMError):
            lbm.lbm_set_geometry(h, None, 7, 8 * 8 * 8)  # unknown wall model
        lbm.lbm_set_geometry(h, None, lbm.LBM_WALL_NODAL, 8 * 8 * 8)  # geometry on a slab is allowed (nz_local + 4 planes)
        plain = lbm.lbm_create(8, 8, 8, 19, 0.8)
        assert lbm.load().lbm_slab_export(plain, None) == lbm.LBM_EINVAL
        with pytest.raises(lbm.LBMError):
            lbm.lbm_slab_export(plain)
        lbm.lbm_destroy(plain)
    finally:
        lbm.lbm_destroy(h)
        lbm.lbm_destroy(other)


# --------------------------------------------------------------------------- two processes, CUDA IPC
IPC_WORKER = r"""
import os, sys, json
import numpy as np
import torch
import torch.distributed as dist
sys.path.insert(0, os.environ["LBM_ROOT"])
from paper_2201_11330_b200 import inputs, lbm, replicas, slabs
rank, local_rank, world = replicas.init(backend="gloo")
torch.cuda.set_device(0)  # both ranks share the one GPU: host-synchronised mode, no rank ever waits on the device
lbm.load()
w = inputs.Workload("ipc", 20, 12, 11, 19, 0.7, 6, face_kind=(0, 0, 1, 1, 0, 0), u0=0.04, noise=1e-3, seed=inputs.SEED_BASE + 9)
g = slabs.SlabSolver(w, rank, world, device_sync=False)
g.init_equilibrium()
torch.cuda.synchronize(); replicas.barrier()
for _ in range(w.steps):
    g.step(1)
    torch.cuda.synchronize(); replicas.barrier()
own = g.get_populations().cpu().view(w.Q, g.nz_local, -1)
tot = slabs.all_reduce_diagnostics(g.diagnostics())
parts = [None] * world
dist.all_gather_object(parts, own.numpy())
if rank == 0:
    f = np.concatenate(parts, axis=1).reshape(w.Q, -1)
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w)
    s.init_equilibrium(torch.from_numpy(rho).cuda(), torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda())
    s.step(w.steps)
    one = s.get_populations().cpu().numpy()
    d1 = s.diagnostics()
    s.close()
    print("OUT" + json.dumps({"equal": bool(np.array_equal(f, one)), "maxdiff": float(np.abs(f - one).max()),
                              "mass_rel": float(abs(tot[0] - d1[0]) / d1[0]), "umax_equal": bool(tot[5] == d1[5])}), flush=True)
replicas.barrier()
g.close()
replicas.finalize()
"""


def test_two_processes_connected_through_cuda_ipc(mods, tmp_path):
    """One process per slab as under torchrun (descriptors exchanged as bytes, neighbour memory opened with CUDA IPC,
    halo planes filled by the other process's kernel).  Both processes share this one GPU, so the run is
    host-synchronised (lbm_slab_set_sync(0)): a step, a stream sync, a barrier."""
    import json
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "ipc_worker.py"
    script.write_text(IPC_WORKER)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, LBM_ROOT=root, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-8000:]
    out = [json.loads(ln[3:]) for ln in r.stdout.splitlines() if ln.startswith("OUT")][-1]
    assert out["equal"], out
    assert out["mass_rel"] <= 1e-13 and out["umax_equal"]


IPC_WORKER_DEVICE_SYNC = IPC_WORKER.replace(
    "g = slabs.SlabSolver(w, rank, world, device_sync=False)", "g = slabs.SlabSolver(w, rank, world, device_sync=True)").replace(
    """for _ in range(w.steps):
    g.step(1)
    torch.cuda.synchronize(); replicas.barrier()
""", """g.step(w.steps)   # all steps in one call, no host synchronisation between them: the two processes are ordered by
# lbm_moments_host between unsynchronised step calls (the neighbour may already be a step ahead and push into the idle
# buffer's halo planes: the host entry points of a slab stage in a scratch allocation, not in that buffer)
r_h = torch.empty(g.N, dtype=torch.float64).pin_memory(); u_h = torch.empty(3 * g.N, dtype=torch.float64).pin_memory()
d_mid = lbm.lbm_moments_host(g.h, r_h, u_h, True)
assert d_mid[7] == 0 and abs(float(r_h.view(g.nz_local + 2, -1)[1:-1].sum()) - d_mid[0]) <= 1e-9 * d_mid[0]
g.step(w.steps)   # the device-side step counters alone (cuStreamWaitValue32 on the neighbour's counter)
torch.cuda.synchronize(); replicas.barrier()
""").replace("s.step(w.steps)\n    one =", "s.step(2 * w.steps)\n    one =")


def test_two_processes_with_device_side_ordering(mods, tmp_path):
    """The same two processes with lbm_slab_set_sync left ON: each rank enqueues all its steps at once, and a step starts
    when the stream's cuStreamWaitValue32 sees the neighbour's counter (written by the OTHER process's slab_signal_kernel
    through CUDA IPC memory).  Two contexts time-share this one GPU; a wait-value is a front-end wait, not a spinning
    kernel, so the waiting context yields and the pair makes progress (measured: 2 x 200 steps in 34 ms).  The worker
    runs under its own process group with a 150 s limit, so a deadlock would fail the test instead of hanging the box."""
    import json
    import os
    import signal
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    assert "device_sync=True" in IPC_WORKER_DEVICE_SYNC and "g.step(w.steps)   # all steps" in IPC_WORKER_DEVICE_SYNC
    assert "s.step(2 * w.steps)" in IPC_WORKER_DEVICE_SYNC
    script = tmp_path / "ipc_worker_device_sync.py"
    script.write_text(IPC_WORKER_DEVICE_SYNC)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, LBM_ROOT=root, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    p = subprocess.Popen(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, start_new_session=True)
    try:
        out, err = p.communicate(timeout=150)
    except subprocess.TimeoutExpired:
        os.killpg(p.pid, signal.SIGKILL)
        p.communicate()
        pytest.fail("two processes ordered by device-side counters made no progress on one GPU within 150 s")
    assert p.returncode == 0, err[-8000:]
    res = [json.loads(ln[3:]) for ln in out.splitlines() if ln.startswith("OUT")][-1]
    assert res["equal"], res
    assert res["mass_rel"] <= 1e-13 and res["umax_equal"]


# --------------------------------------------------------------------------- solid masks, nodal walls, mirror planes on slabs
def _oracle_geo_run(w, steps):
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force, face_rho=w.face_rho)
    if w.has_geometry:
        o.set_geometry(w.geo(), w.wall_model)
    for k, prof in w.face_profiles().items():
        o.set_face_velocity(k, prof)
    o.init_equilibrium(rho, u)
    o.step(steps)
    out = o.get_f(), o.boundary_force() if w.has_geometry else None
    o.close()
    return out


class _Lumpy(inputs.Workload):
    """A workload whose mask has bodies next to every cut of a 2- / 3- / 4-slab split, on the z faces and single nodes."""

    def geo(self):
        nx, ny, nz = self.nx, self.ny, self.nz
        g = inputs.sphere_mask(nx, ny, nz, (0.4 * nx, 0.5 * ny, 0.5 * nz), 0.3 * min(nx, ny, nz)).reshape(nz, ny, nx).copy()
        g[0:2, 1:4, 2:5] = 1            # a block on the z- face
        g[nz - 1, ny - 3:, nx - 4:] = 1  # a plate in the last plane
        for z in range(nz):             # a thin diagonal rod through every plane
            g[z, (2 + z) % ny, (nx - 2 - z) % nx] = 1
        return g.reshape(-1)

    @property
    def has_geometry(self):
        return True


def _lumpy(dims, Q, tau, model, faces, eq=EQ_STANDARD, force=(0.0, 0.0, 0.0), steps=9):
    S_, PR_ = inputs.FACE_SYMMETRY, inputs.FACE_PRESSURE
    fu = np.zeros((6, 3))
    for k in range(6):
        if faces[k] == M:
            fu[k] = (0.03, 0.0, 0.01 if k < 4 else 0.0)
    return _Lumpy(f"lumpy_{Q}_{model}", dims[0], dims[1], dims[2], Q, tau, steps, face_kind=tuple(faces),
                  face_u=tuple(map(tuple, fu)), force=tuple(force), noise=1e-3, seed=inputs.SEED_BASE + 91, kind="rest",
                  eq=eq, wall_model=model, face_rho=(1.0, 0.99, 1.0, 1.0, 1.01, 0.98))


_S, _PR = inputs.FACE_SYMMETRY, inputs.FACE_PRESSURE
GEO_CASES = {
    "periodic_q19_forced": dict(dims=(20, 12, 12), Q=19, tau=0.8, faces=[P] * 6, force=(1e-5, 0, 2e-6)),
    "zwalls_q27": dict(dims=(14, 10, 13), Q=27, tau=0.7, faces=[P, P, P, P, B, B], force=(2e-5, 0, 0)),
    "sphere_case_faces_q27": dict(dims=(22, 8, 12), Q=27, tau=0.6, faces=[M, _PR, _S, _S, P, P], eq=EQ_INCOMP),
    "open_z_mirror_x_q19": dict(dims=(10, 9, 14), Q=19, tau=0.66, faces=[_S, _S, B, B, M, _PR]),
}


@pytest.mark.parametrize("nslabs", [2, 3, 4])
@pytest.mark.parametrize("model", [inputs.WALL_HALFWAY, inputs.WALL_NODAL], ids=["halfway", "nodal"])
@pytest.mark.parametrize("case", list(GEO_CASES))
def test_slabs_with_geometry_equal_the_undivided_box(mods, case, model, nslabs):
    """lbm_set_geometry on slab handles (mask with two halo planes per side): solid bodies across the cuts, nodal wall
    nodes in the halo planes, mirror planes and open faces — bit-identical to the undivided CUDA run, 1e-12 from the
    oracle, and the slabs' parts of Eq. 13 add up to the whole force."""
    lbm, slabs = mods
    w = _lumpy(model=model, **GEO_CASES[case])
    ref, Fref = _oracle_geo_run(w, w.steps)
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w)
    s.init_equilibrium(torch.from_numpy(rho).cuda(), torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda())
    s.step(w.steps)
    one = s.get_populations().clone()
    F1 = s.boundary_force()
    s.close()
    assert float(np.abs(one.cpu().numpy() - ref).max()) <= TOL
    g = slabs.SlabGroup(w, nslabs)
    g.init_equilibrium()
    g.step(w.steps)
    f = g.get_populations()
    F = g.boundary_force()
    g.close()
    assert torch.equal(f, one), f"{case}: slabs differ from the undivided CUDA run by {float((f - one).abs().max())}"
    assert np.abs(F - F1).max() <= 1e-12 * max(1.0, np.abs(F1).max())
    assert np.abs(F - Fref).max() <= 1e-12 * max(1.0, np.abs(Fref).max())


def test_sphere_case_on_slabs(mods):
    """inputs.config(8) (the paper's sphere case with its boundaries) shrunk by 4, cut into 4 slabs: the cut
    at z = 16 goes through the sphere."""
    lbm, slabs = mods
    w = inputs.config(8).shrunk(4, steps=60)
    ref, Fref = _oracle_geo_run(w, w.steps)
    g = slabs.SlabGroup(w, 4)
    g.init_equilibrium()
    g.step(w.steps)
    f = g.get_populations().cpu().numpy()
    F = g.boundary_force()
    g.close()
    assert np.abs(f - ref).max() <= TOL
    assert np.abs(F - Fref).max() <= 1e-12
