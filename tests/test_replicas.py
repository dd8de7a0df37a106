"""world_size-2 gloo test (CPU) of the only multi-process logic in the path: bench.py --gpus N runs
independent replicas; the whole-job value is (sum of cell updates) / (max over ranks of device time)."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["LBM_ROOT"])
from paper_2201_11330_b200 import replicas
rank, local_rank, world = replicas.init(backend="gloo")
assert world == 2 and rank == local_rank
replicas.barrier()
secs = 2.0 if rank == 0 else 3.5          # the slower rank defines the job time
units, tmax, ups = replicas.aggregate_throughput(1000.0 * (rank + 1), secs)
mx = replicas.max_over_ranks(float(rank))
replicas.barrier()
if rank == 0:
    print(json.dumps({"units": units, "tmax": tmax, "ups": ups, "mx": mx}))
replicas.finalize()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_replica_aggregation_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, LBM_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [ln for ln in r.stdout.splitlines() if ln.startswith("{")][-1]
    out = json.loads(line)
    assert out["units"] == 3000.0 and out["tmax"] == 3.5 and out["mx"] == 1.0
    assert out["ups"] == pytest.approx(3000.0 / 3.5)


def test_single_process_is_identity():
    from paper_2201_11330_b200 import replicas
    assert replicas.env_world() == (0, 0, 1) or "RANK" in os.environ
    assert replicas.max_over_ranks(1.25) == 1.25
    assert replicas.aggregate_throughput(10.0, 2.0) == (10.0, 2.0, 5.0)


def test_reference_arm_runs_on_cpu():
    """bench.py --impl reference times the oracle on host cores and prints the contract's JSON line."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "2", "--warmup", "1",
                        "--config", "0"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    out = json.loads(r.stdout.strip().splitlines()[-1])
    assert out["impl"] == "reference" and out["unit"] == "MLUPS" and out["value"] > 0
    assert out["cpu_baseline"]["kind"] == "oracle" and out["e2e"]["h2d_bytes_per_step"] == 0
