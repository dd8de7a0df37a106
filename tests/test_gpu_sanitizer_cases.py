"""Every kernel variant of the library once, on grids of at most 32^3, each compared with the CPU oracle — the subset
that is run under compute-sanitizer (SURVEY.md section 4 T4, section 5 "race detection"):

    compute-sanitizer --tool memcheck  --error-exitcode 1 python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q -x
    compute-sanitizer --tool racecheck --error-exitcode 1 python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q -x
    compute-sanitizer --tool initcheck --error-exitcode 1 python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q -x
    compute-sanitizer --tool synccheck --error-exitcode 1 python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q -x

(one tool per GPU-box call; PYTORCH_NO_CUDA_MEMORY_CACHING=1 gives every tensor its own allocation so that memcheck sees
the bounds of the caller's arrays too).  On the pool this was written on compute-sanitizer is closed (profiles/sanitizer_r02.md
has the answer it gives), so every case here also runs the library's own stand-ins (include/lbm.h "Debug aids"):
lbm_debug_arm(poison) fills every population / scratch array with NaNs before the initialisation — a value computed from
a slot nobody wrote fails the comparison with the oracle — and lbm_debug_check verifies the guard zones around every
device array afterwards (an out-of-bounds store).  Two negative tests prove that both alarms ring.  Without a sanitizer
it is an ordinary `-m gpu` parity test file (a few seconds).

Covered: stream_collide_ab (periodic / walls / link mask, forcing, fp32 storage, mirror planes), stream_collide_aa_even /
_odd, stream_collide_ab_persistent, stream_collide_aa_persistent, init_equilibrium (device and host entry points),
import_canonical / export_canonical, moments_kernel + reduce_final_kernel (device and host entry points),
classify_nodes_kernel / build_links_kernel through lbm_set_geometry and lbm_set_geometry_host (staging), halfway and
nodal walls, boundary_force_kernel, open faces (inlet profile, pressure outlet), z-slabs in one process (peer pushes,
slab_signal_kernel, stream waits) with and without a mask.
"""
import numpy as np
import pytest

from oracle import Oracle
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


def oracle_of(w):
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau, eq=w.eq, face_kind=w.face_kind, face_u=w.face_u, force=w.force, face_rho=w.face_rho)
    if w.has_geometry:
        o.set_geometry(w.geo(), w.wall_model)
    for face, prof in w.face_profiles().items():
        o.set_face_velocity(face, prof)
    return o


def workloads():
    lid = tuple((0.0, 0.0, 0.0) for _ in range(5)) + ((0.1, 0.0, 0.0),)
    return {
        "tgv_q19": inputs.config(0).scaled(20, steps=5),
        "cavity_q19": inputs.config(2).scaled(18, steps=5),
        "channel_q27_forced": inputs.Workload("san_channel", 21, 10, 9, 27, 0.9, 5, face_kind=(P, P, P, P, B, B), force=(1e-5, 0.0, 2e-6),
                                              noise=1e-4, seed=7, kind="rest"),
        "mixed_q19_incomp": inputs.Workload("san_mixed", 19, 11, 8, 19, 0.7, 5, face_kind=(B, M, P, P, M, B),
                                            face_u=((0, 0, 0), (0.0, 0.03, -0.02), (0, 0, 0), (0, 0, 0), (0.05, 0.01, 0.0), (0, 0, 0)),
                                            noise=1e-4, seed=8, kind="rest", eq=inputs.EQ_INCOMP),
        "d2q9_tgv": inputs.Workload("san_d2q9", 40, 24, 2, 9, 0.7, 5, u0=0.03, noise=1e-4, seed=9),
        "sphere_nodal_q27": inputs.config(5).shrunk(8, steps=5),           # 64 x 16 x 16, link mask, nodal, forced, Eq. 5
        "sphere_halfway_q19": inputs.Workload("san_sphere_hw", 24, 16, 14, 19, 0.8, 5, face_kind=(P, P, B, B, B, M), face_u=lid,
                                              noise=1e-4, seed=10, kind="rest", sphere=(9.0, 8.0, 7.0, 3.2)),
        "sphere_open_sym_q27": inputs.config(8).shrunk(8, steps=5),        # inlet / outlet / mirror planes + nodal sphere
        "cylinder_q9_open": inputs.config(7).shrunk(4, steps=5),           # D2Q9 inlet profile + pressure outlet + mask
    }


WL = workloads()


def run_single(lbm, w, scheme, store, persistent, host_entry):
    rho, u = w.fields()
    uf = np.ascontiguousarray(u.reshape(-1))
    s = lbm.Solver.from_workload(w, scheme=scheme, store=store)
    s.set_persistent(persistent)
    s.debug_arm(poison=True)  # NaNs in every population / scratch array: a slot used before it is written shows up below
    if host_entry:
        s.init_equilibrium_host(torch.from_numpy(rho), torch.from_numpy(uf))
    else:
        s.init_equilibrium(torch.from_numpy(rho).cuda(), torch.from_numpy(uf).cuda())
    f0 = s.get_populations().cpu().numpy()
    s.step(w.steps)
    f = s.get_populations().cpu().numpy()
    if host_entry:
        r_h, u_h = torch.empty(w.N, dtype=torch.float64), torch.empty(3 * w.N, dtype=torch.float64)
        d = lbm.lbm_moments_host(s.h, r_h, u_h, True)
        r, uu = r_h.numpy(), u_h.numpy().reshape(3, -1)
    else:
        r_d, u_d, d = s.moments()
        r, uu = r_d.cpu().numpy(), u_d.cpu().numpy()
    F = s.boundary_force() if w.has_geometry and w.geo() is not None else None
    # checkpoint round trip: export, import, one more step
    s.set_populations(torch.from_numpy(f.reshape(-1)).cuda())
    s.step(1)
    f1 = s.get_populations().cpu().numpy()
    torch.cuda.synchronize()
    assert s.debug_check() == 0, "a kernel stored outside an array (guard zone damaged)"
    s.close()
    return f0, f, r, uu, d, F, f1


# (mirror planes need the A/B scheme, include/lbm.h)
VARIANTS = [(n, s, p) for n in WL for s in ("ab", "aa") for p in (1, 0) if not (s == "aa" and inputs.FACE_SYMMETRY in WL[n].face_kind)]


@pytest.mark.parametrize("name,scheme,persistent", VARIANTS)
def test_every_variant_against_the_oracle(mods, name, scheme, persistent):
    lbm, _ = mods
    w = WL[name]
    o = oracle_of(w)
    rho, u = w.fields()
    o.init_equilibrium(rho, u)
    ref0 = o.get_f()
    o.step(w.steps)
    ref = o.get_f()
    ro, uo, do = o.moments()
    Fo = o.boundary_force() if w.has_geometry and w.geo() is not None else None
    o.step(1)
    ref1 = o.get_f()
    o.close()
    f0, f, r, uu, d, F, f1 = run_single(lbm, w, {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme], lbm.LBM_STORE_F64,
                                        persistent, host_entry=(persistent == 0))
    assert np.abs(f0 - ref0).max() <= 1e-15
    assert np.abs(f - ref).max() <= TOL
    assert np.abs(f1 - ref1).max() <= TOL
    assert np.abs(r - ro).max() <= 1e-13 and np.abs(uu - uo).max() <= 1e-13
    np.testing.assert_allclose(d[:5], do[:5], rtol=1e-12, atol=1e-12)
    assert d[7] == do[7] == 0
    if Fo is not None:
        assert np.abs(F - Fo).max() <= 1e-12


@pytest.mark.parametrize("scheme", ["ab", "aa"])
@pytest.mark.parametrize("name", ["tgv_q19", "cavity_q19", "channel_q27_forced", "sphere_nodal_q27", "cylinder_q9_open"])
def test_fp32_storage_variants(mods, name, scheme):
    lbm, _ = mods
    w = WL[name]
    o = oracle_of(w)
    rho, u = w.fields()
    o.init_equilibrium(rho, u)
    o.step(w.steps)
    ref = o.get_f()
    o.close()
    _, f, _, _, d, _, _ = run_single(lbm, w, {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme], lbm.LBM_STORE_F32, 0, False)
    t = np.abs(ref).max(axis=1, keepdims=True)
    assert (np.abs(f - ref) / t).max() <= 2e-5 and d[7] == 0


@pytest.mark.parametrize("store", ["f64", "f32"])
@pytest.mark.parametrize("name,nslabs", [("tgv_q19", 3), ("cavity_q19", 2), ("channel_q27_forced", 3), ("sphere_nodal_q27", 2),
                                         ("sphere_open_sym_q27", 2)])
def test_slabs_in_one_process(mods, name, nslabs, store):
    """Peer pushes into the neighbours' halo planes, slab_signal_kernel and the stream waits (all slabs on one device)."""
    lbm, slabs = mods
    w = WL[name]
    o = oracle_of(w)
    rho, u = w.fields()
    o.init_equilibrium(rho, u)
    o.step(w.steps)
    ref = o.get_f()
    Fo = o.boundary_force() if w.has_geometry else None
    o.close()
    g = slabs.SlabGroup(w, nslabs, store=lbm.LBM_STORE_F32 if store == "f32" else lbm.LBM_STORE_F64)
    for sl in g.slabs:
        lbm.lbm_debug_arm(sl.h, True)
    g.init_equilibrium()
    g.step(w.steps)
    f = g.get_populations().cpu().numpy()
    d = g.diagnostics()
    F = g.boundary_force() if w.has_geometry else None
    g.synchronize()
    assert [lbm.lbm_debug_check(sl.h) for sl in g.slabs] == [0] * nslabs
    g.close()
    if store == "f64":
        assert np.abs(f - ref).max() <= TOL
        if Fo is not None:
            assert np.abs(F - Fo).max() <= 1e-12
    else:
        assert (np.abs(f - ref) / np.abs(ref).max(axis=1, keepdims=True)).max() <= 2e-5
    assert d[7] == 0


def test_guard_zones_detect_an_out_of_bounds_store(mods):
    """The alarm rings: one byte written just outside a population buffer (its address comes from the slab descriptor)
    is counted by lbm_debug_check; nothing is counted before, nothing after re-arming."""
    lbm, _ = mods
    runtime = pytest.importorskip("cuda.bindings.runtime")
    h = lbm.lbm_create_slab(16, 8, 4, 0, 4, 19, 0.8)
    try:
        assert lbm.lbm_debug_check(h) == 0
        d = lbm.lbm_slab_export(h)
        nbytes = 19 * 16 * 8 * 6 * 8
        for addr in (int(d.buf[0]) - 1, int(d.buf[1]) + nbytes):  # one byte before buffer 0, one byte after buffer 1
            (err,) = runtime.cudaMemset(addr, 0, 1)
            assert int(err) == 0
        torch.cuda.synchronize()
        assert lbm.lbm_debug_check(h) == 2
        lbm.lbm_debug_arm(h, False)
        assert lbm.lbm_debug_check(h) == 0
    finally:
        lbm.lbm_destroy(h)


def test_poison_makes_an_uninitialised_read_visible(mods):
    """The alarm rings: poisoned and NOT initialised, every cell reports non-finite moments; after the initialisation
    (which must overwrite every slot a step reads) none does, through steps of both schemes."""
    lbm, _ = mods
    for scheme in (lbm.LBM_SCHEME_AB, lbm.LBM_SCHEME_AA):
        s = lbm.Solver(12, 10, 8, 19, 0.8, scheme=scheme, face_kind=[B, B, P, P, B, M], face_u=[[0, 0, 0]] * 5 + [[0.05, 0, 0]])
        s.debug_arm(poison=True)
        assert s.diagnostics()[7] == 12 * 10 * 8
        s.init_equilibrium()
        s.set_persistent(0)
        s.step(3)
        assert s.diagnostics()[7] == 0
        s.close()
