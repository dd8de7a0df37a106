"""The bench.py contract on a GPU box: one JSON line with the keys the driver reads, for the device-resident number, the
end-to-end number through the host-buffer C-ABI calls, the roofline object and the CPU baseline (oracle) — on the small
config 1 (128^3) so that it runs in seconds.  The numbers themselves are not judged here."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*args):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_has_the_contract_keys():
    d = _run("--config", "1", "--steps", "50", "--warmup", "3")
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["unit"] == "MLUPS" and d["dtype"] == "f64" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["n_gpus"] == 1 and d["steps"] == 50 and d["warmup"] >= 3 and d["higher_is_better"] is True
    assert d["config"]["workload"] == "cfg1_q19_tgv128" and "model" not in d["config"]
    # nothing but the fused kernel is timed: periodic D3Q19 fp64 takes two time steps per launch (stream_collide_ab2)
    assert d["gpu_launches"] == 25 and d["roofline"]["steps_per_launch"] == 2
    one = _run("--config", "1", "--steps", "50", "--warmup", "3", "--two-step", "0", "--no-cpu-baseline")
    assert one["gpu_launches"] == 50 and one["roofline"]["steps_per_launch"] == 1  # one launch per time step
    assert abs(d["value"] - 128**3 * 50 / (d["ms_per_step"] * 50 * 1e-3) / 1e6) <= 1e-6 * d["value"]
    r = d["roofline"]
    assert r["bound"] == "hbm" and r["unit"] == "GB/s" and r["bytes_per_cell_update"] == 304
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12
    assert abs(r["achieved"] - d["value"] * 1e6 * 304 / 1e9) <= 1e-6 * r["achieved"]
    # what the launch itself must move (one read + one write of every population per launch, one step or two) and what ncu
    # saw it move can never be much above the measured peak — `frac` may be (two steps per pass), these two may not
    for rr, spl in ((r, 2), (one["roofline"], 1)):
        assert rr["floor_bytes_per_launch"] == 304 * 128**3
        assert abs(rr["floor_frac"] - rr["frac"] / spl) <= 1e-9 * rr["floor_frac"]
        assert 0 < rr["floor_frac"] <= 1.2
        assert rr["dram_frac"] is None or 0 < rr["dram_frac"] <= 1.2
    e = d["e2e"]
    assert e["unit"] == "MLUPS" and 0 < e["value"] < d["value"] and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["unit"] == "MLUPS" and c["cores"] >= 1 and 0 < c["value"] < d["value"]
    assert d["checks"]["nonfinite_cells"] == 0 and d["checks"]["mass_drift_rel"] < 1e-12


def test_bench_runs_the_papers_examples():
    for cfg, name in ((7, "cfg7_q9_cylinder512x128"), (8, "cfg8_q27_sphere_open512x128x128")):
        d = _run("--config", str(cfg), "--steps", "30", "--warmup", "3", "--no-cpu-baseline")
        # cfg7 (65 536 cells) fits the device at once: all 30 steps in one launch of the persistent kernel
        assert d["config"]["workload"] == name and d["gpu_launches"] == (1 if cfg == 7 else 30) and d["checks"]["nonfinite_cells"] == 0
        assert d["roofline"]["steps_per_launch"] == 30 / d["gpu_launches"]
        assert d["roofline"]["bytes_per_cell_update"] == 2 * (9 if cfg == 7 else 27) * 8 + 4  # + the 4-byte link mask
        if cfg == 7:  # persistent kernel on an L2-resident grid: no HBM floor is claimed
            assert d["roofline"]["floor_frac"] is None and d["roofline"]["dram_frac"] is None
        else:
            assert 0 < d["roofline"]["floor_frac"] <= 1.2 and 0 < d["roofline"]["dram_frac"] <= 1.2
