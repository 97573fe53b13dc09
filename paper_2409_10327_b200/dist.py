"""Multi-GPU plumbing for the benchmark: the renderer itself is one-GPU (BASELINE.json north_star: no sharding, no
collectives), so N > 1 means N independent replicas, one frame per rank.  The only cross-rank traffic is the timing
protocol: a barrier on both sides of the timed region and the MAX over ranks of the device time."""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def barrier() -> None:
    if world()[1] > 1:
        dist.barrier()


def max_over_ranks(ms: float, device="cpu") -> float:
    """Slowest rank's time: the job is as fast as its slowest replica."""
    if world()[1] == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, ms_max: float) -> float:
    """Aggregate units/s over all replicas (weak scaling: per-rank work is fixed)."""
    return world()[1] * units_per_rank / (ms_max * 1e-3)
