"""N > 1 launches (torchrun, one process per GPU): "replicas only".

BASELINE.json's north_star fixes one GPU with no sharding and no collectives, so the path does not shard in this
build: under `bench.py --gpus N` every rank advances its own replica of the workload and no
data-path collective exists.  What remains is host logic: the barrier around the timed region, the max over ranks of
the device-side time, and the whole-job throughput.  It holds none of the method's arithmetic.
"""
from __future__ import annotations

import os


def dist_env():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) for a plain launch."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def barrier(world: int) -> None:
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(ms: float, world: int, device: str = "cpu") -> float:
    """The timed region of a job is as long as its slowest rank."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(points_per_rank: int, cn_steps: int, ms: float, world: int) -> float:
    """Gpoint-steps/s of all replicas together ("weak" scaling: per-GPU work is fixed as N grows)."""
    return world * points_per_rank * cn_steps / (ms * 1e-3) / 1e9
