"""BASELINE.json configs 3-5 at their FULL step counts on the GPU (2000 / 200 / 20000 steps): no oracle can follow at
these sizes, so the checks are the ones that hold at any size — conservation, symmetry, the analytic start-up solution.
About 4 minutes of GPU time, therefore opt-in:  LBM_FULL_LENGTH=1 python -m pytest tests/test_gpu_full_length.py -m gpu -s
(the shorter versions of the same checks run in tests/test_gpu_parity.py on every `pytest -m gpu`)."""
import os
import time

import numpy as np
import pytest

from paper_2201_11330_b200 import inputs

pytestmark = [pytest.mark.gpu, pytest.mark.skipif(os.environ.get("LBM_FULL_LENGTH") != "1", reason="opt-in: LBM_FULL_LENGTH=1")]
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
