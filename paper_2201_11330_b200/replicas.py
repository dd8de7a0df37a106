"""Host-side plumbing for `bench.py --gpus N`: the path does not shard in this build (BASELINE.json
north_star: one GPU, no collectives), so N ranks run N independent replicas of the workload
("replicas only").  The only cross-rank traffic is the barrier around the timed
region and the MAX-reduction of the per-rank device time.  Works with the nccl backend on GPUs
and with gloo on CPU (tests/test_replicas.py, world_size 2).
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if unset)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str | None = None):
    """Join the process group if launched under torchrun with WORLD_SIZE > 1.  Returns
    (rank, local_rank, world_size)."""
    rank, local_rank, world = env_world()
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX of a per-rank scalar (the per-rank device time of the timed region)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu"):
    """Whole-job throughput of independent replicas: (sum of units over ranks) / (max time over ranks).
    Returns (units_total, seconds_max, units_per_second)."""
    units = sum_over_ranks(units_this_rank, device)
    secs = max_over_ranks(seconds_this_rank, device)
    return units, secs, units / secs


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
