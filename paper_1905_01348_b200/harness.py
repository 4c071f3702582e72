"""Host-side helpers of the benchmark harness (no arithmetic of the method).

The path is single-GPU by construction (BASELINE.json north_star: "one GPU, with no sharding or
collectives"), so N > 1 means N independent replicas ("replicas only"): each rank runs the
same step on its own device, and the job's throughput is the work of all ranks over the slowest
rank's device time.  The only cross-rank traffic is the barrier and this MAX reduction of a timing.
"""
from __future__ import annotations


def dist_or_none():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX of a host scalar over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    dist = dist_or_none()
    if dist is None:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(units_per_rank: float, seconds_this_rank: float, device="cpu") -> float:
    """Whole-job units/s of world_size replicas: world * units / max_r(seconds_r)."""
    dist = dist_or_none()
    world = dist.get_world_size() if dist is not None else 1
    return world * units_per_rank / max_over_ranks(seconds_this_rank, device)


def barrier(device=None):
    import torch
    dist = dist_or_none()
    if dist is not None:
        dist.barrier()
    if device is not None and torch.cuda.is_available():
        torch.cuda.synchronize(device)
