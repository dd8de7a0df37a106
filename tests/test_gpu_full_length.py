"""BASELINE.json configs 3-5 at their FULL step counts on the GPU (2000 / 200 / 20000 steps).  No oracle can follow a
512^3 box directly, so the checks are (i) the ones that hold at any size — conservation, symmetry, the analytic start-up
solution — and (ii) for the headline config an every-cell, full-length parity CHAIN: the 512^3 box started from a 128^3
field tiled 4 x 4 x 4 must equal the 128^3 CUDA run tile by tile, bit for bit, after all 200 steps, and that 128^3 run
must match the oracle to 1e-12 in the same test.  About 4 minutes of GPU time in total (the 20000-step channel is 170 s);
part of every `pytest -m gpu`."""
import time

import numpy as np
import pytest

from paper_2201_11330_b200 import inputs

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def lbm():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2201_11330_b200 import lbm as _lbm
    _lbm.load()
    return _lbm


def _run(lbm, w, sample_every=None):
    rho, u = w.fields()
    s = lbm.Solver.from_workload(w, scheme=lbm.LBM_SCHEME_AB)
    s.init_equilibrium_host(torch.from_numpy(rho).pin_memory(), torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).pin_memory())
    d0 = s.diagnostics()
    hist = [(0, d0[4])]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    done = 0
    while done < w.steps:
        n = min(sample_every or w.steps, w.steps - done)
        s.step(n)
        done += n
        if sample_every:
            hist.append((done, s.diagnostics()[4]))
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    print(f"\n{w.name}: {w.steps} steps in {dt:.1f} s = {w.N * w.steps / dt / 1e6:.0f} MLUPS (host clock, diagnostics included)")
    return s, d0, hist


def test_config3_tgv512_energy_history(lbm):
    """BJ configs[3]: 512^3 Taylor-Green, tau 0.52, 200 steps: mass and momentum conserved to round-off, the kinetic
    energy falls monotonically (Re ~ 489: only reported against the viscous-limit rate, R11)."""
    w = inputs.config(3)
    s, d0, hist = _run(lbm, w, sample_every=20)
    d = s.diagnostics()
    s.close()
    assert abs(d[0] - d0[0]) <= 1e-12 * d0[0] and d[7] == 0
    # the momentum the seeded density noise starts with (sum rho u ~ 1e-2 of 1.3e8 cells) stays what it was
    assert max(abs(d[k] - d0[k]) for k in (1, 2, 3)) <= 1e-9
    e = np.array([h[1] for h in hist])
    assert (np.diff(e) < 0).all()
    nu, k2 = (w.tau - 0.5) / 3, 3 * (2 * np.pi / 512) ** 2
    print("E(t)/E(0):", " ".join(f"{v / e[0]:.5f}" for v in e), f"| viscous limit exp(-2 nu k^2 t) at t = 200: {np.exp(-2 * nu * k2 * 200):.5f}")


def test_config2_cavity256_full_length(lbm):
    """BJ configs[2]: 256^3 lid-driven cavity, 2000 steps: total mass constant (the lid's +- links cancel, R6), u_y
    antisymmetric and u_x symmetric under the y-mirror (started noise-free)."""
    w = inputs.config(2)
    s, d0, _ = _run(lbm, w)
    rho, u, d = s.moments()
    s.close()
    n = w.nx
    assert abs(d[0] - d0[0]) <= 1e-11 * d0[0] and d[7] == 0
    ux, uy = u[0].view(n, n, n), u[1].view(n, n, n)
    assert float((uy + uy.flip(1)).abs().max()) <= 1e-12
    assert float((ux - ux.flip(1)).abs().max()) <= 1e-12
    assert 0.05 < d[5] <= 0.1 + 1e-9  # the lid drags the fluid, nothing exceeds the lid speed
    print(f"cavity: max|u| = {d[5]:.5f}, relative mass drift {abs(d[0] - d0[0]) / d0[0]:.2e}")


def test_config4_channel512_full_length(lbm):
    """BJ configs[4]: D3Q27 512^3 forced channel, 20000 steps: the plane-averaged u_x(z) against the analytic start-up
    series (R9: H^2/(pi^2 nu) = 199 000 steps, so 20000 steps is not the steady parabola) to 1e-3 relative L2."""
    w = inputs.config(4)
    s, d0, _ = _run(lbm, w)
    _, uf, d = s.moments()
    s.close()
    prof = uf[0].view(512, 512 * 512).mean(dim=1).cpu().numpy()
    H, F, nu, steps = 512, w.force[0], (w.tau - 0.5) / 3, w.steps
    z = np.arange(H) + 0.5
    u_an = F * z * (H - z) / (2 * nu)
    for n_ in range(1, 4000, 2):
        u_an -= 4 * F * H * H / (nu * np.pi**3 * n_**3) * np.sin(n_ * np.pi * z / H) * np.exp(-n_ * n_ * np.pi**2 * nu * steps / H**2)
    err = np.linalg.norm(prof - u_an) / np.linalg.norm(u_an)
    print(f"channel: centreline u_x = {prof[256]:.6e} (series {u_an[256]:.6e}), rel. L2 error of the profile {err:.2e}")
    assert err < 1e-3
    assert abs(d[0] / w.N - 1) < 1e-5 and d[7] == 0


@pytest.mark.parametrize("scheme", ["ab", "aa"])
def test_config3_tgv512_every_cell_full_length_chain(lbm, scheme):
    """BJ configs[3] parameters (tau 0.52, u0 0.04, noise 1e-4, 200 steps) on a 128^3 periodic box: the CUDA run equals the
    oracle to 1e-12 over the whole field; the SAME field tiled 4 x 4 x 4 over the 512^3 box of the headline run (the launch
    configuration bench.py times) then gives, after the full 200 steps, the 128^3 populations in every one of the 64
    tiles, bit for bit (a periodic flow whose period divides the box evolves like the small periodic box: same
    arithmetic per cell).  Every cell of the 512^3 run is thereby tied to the oracle at full length."""
    from oracle import Oracle
    n, k = 128, 4
    w = inputs.config(3).scaled(n)  # same tau, u0, noise amplitude and seed as configs[3]
    steps = inputs.config(3).steps
    assert (w.tau, w.u0, w.noise, steps) == (0.52, 0.04, 1e-4, 200)
    sch = {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[scheme]
    rho, u = w.fields()
    rho_s = torch.from_numpy(rho).cuda()
    u_s = torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda()
    s = lbm.Solver.from_workload(w, scheme=sch)
    s.init_equilibrium(rho_s, u_s)
    s.step(steps)
    f_small = s.get_populations().clone()
    d_small = s.diagnostics()
    s.close()
    o = Oracle(n, n, n, w.Q, w.tau)
    o.init_equilibrium(rho, u)
    o.step(steps)
    err = float(np.abs(f_small.cpu().numpy() - o.get_f()).max())
    o.close()
    assert err <= 1e-12, err
    N = n * k
    big = lbm.Solver(N, N, N, 19, w.tau, scheme=sch)
    big.debug_arm(poison=True)  # NaNs everywhere before the initialisation; guard zones checked after the run
    rho_b = rho_s.view(n, n, n).repeat(k, k, k).reshape(-1)
    u_b = u_s.view(3, n, n, n).repeat(1, k, k, k).reshape(-1)
    big.init_equilibrium(rho_b, u_b)
    del rho_b, u_b
    big.step(steps)
    d_big = big.diagnostics()
    f_big = big.get_populations()
    assert big.debug_check() == 0
    big.close()
    same = f_big.view(19, k, n, k, n, k, n) == f_small.view(19, 1, n, 1, n, 1, n)
    assert bool(same.all()), f"{int((~same).sum())} of {same.numel()} populations differ from the 128^3 tile"
    assert d_big[7] == 0 and d_big[5] == d_small[5] and d_big[6] == d_small[6]
    print(f"\n512^3 {scheme}: all {same.numel()} populations equal the 128^3 tile after {steps} steps; 128^3 vs oracle max|df| = {err:.2e}")


def test_config1_tgv128_fp32_storage_full_length(lbm):
    """BJ configs[1] (128^3, tau 0.6, 1000 steps) with fp32 storage against the oracle: <= 2e-5 relative (north_star)."""
    from oracle import Oracle
    w = inputs.config(1)
    rho, u = w.fields()
    o = Oracle(w.nx, w.ny, w.nz, w.Q, w.tau)
    o.init_equilibrium(rho, u)
    o.step(w.steps)
    ref = o.get_f()
    o.close()
    for sch in (lbm.LBM_SCHEME_AB, lbm.LBM_SCHEME_AA):
        s = lbm.Solver.from_workload(w, scheme=sch, store=lbm.LBM_STORE_F32)
        s.init_equilibrium(torch.from_numpy(rho).cuda(), torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda())
        s.step(w.steps)
        got = s.get_populations().cpu().numpy()
        s.close()
        rel = float((np.abs(got - ref) / np.abs(ref)).max())
        print(f"\ncfg1 fp32 storage, scheme {sch >> 12}: max relative |df| = {rel:.2e}")
        assert rel <= 2e-5


@pytest.mark.parametrize("name", ["periodic_q19", "cavity_q19", "channel_q27"])
def test_two_steps_per_pass_equal_single_steps_over_a_long_run(lbm, name):
    """Soak test of stream_collide_ab2's shared-memory hand-over (stage 1 of plane k+1 may overlap stage 2 of plane k; the
    ghost planes of the D3Q27 channel): 400 steps on 256 x 256 x 128 cells — every SM busy, thousands of barrier
    crossings per block — must give the same bits as 400 launches of the one-step kernel, and conserve mass."""
    B, M, P = inputs.FACE_BOUNCE, inputs.FACE_MOVING, inputs.FACE_PERIODIC
    lid = tuple((0.0, 0.0, 0.0) for _ in range(5)) + ((0.1, 0.0, 0.0),)
    w = {
        "periodic_q19": inputs.Workload("soak_p", 256, 256, 128, 19, 0.52, 400, u0=0.04, noise=1e-4, seed=inputs.SEED_BASE + 41),
        "cavity_q19": inputs.Workload("soak_c", 256, 256, 128, 19, 0.55, 400, face_kind=(B, B, B, B, B, M), face_u=lid, noise=1e-4,
                                      seed=inputs.SEED_BASE + 42, kind="rest"),
        "channel_q27": inputs.Workload("soak_q27", 256, 256, 128, 27, 0.9, 400, face_kind=(P, P, P, P, B, B), force=(1e-6, 0.0, 0.0),
                                       noise=1e-4, seed=inputs.SEED_BASE + 43, kind="rest"),
    }[name]
    rho, u = w.fields()
    rho_d = torch.from_numpy(rho).cuda()
    u_d = torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).cuda()
    out = []
    for mode in (1, 0):
        s = lbm.Solver.from_workload(w, scheme=lbm.LBM_SCHEME_AB)
        s.set_two_step(mode)
        s.init_equilibrium(rho_d, u_d)
        d0 = s.diagnostics()
        l0 = s.launches
        s.step(w.steps)
        launches = s.launches - l0
        out.append((s.get_populations().clone(), s.diagnostics(), launches))
        s.close()
    assert out[0][2] == w.steps // 2 and out[1][2] == w.steps
    assert torch.equal(out[0][0], out[1][0])
    assert abs(out[0][1][0] - d0[0]) <= 1e-11 * d0[0] and out[0][1][7] == 0
