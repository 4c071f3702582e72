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


# ---- j-sharding over GPUs (the paper's band-index scheme) -----------
# Targets j (and out_j) are partitioned over the ranks; every rank needs all of Phi, so the one exchange step is an
# all-gather of Phi (the paper broadcasts psi_i band by band in fp32).  No reduction is needed: the
# outputs are disjoint.  The benchmark headline stays "replicas only" (BASELINE.json north_star); this is the natural
# multi-GPU form of the operator for when Phi itself is distributed.
def shard_range(n: int, world: int, rank: int):
    """[lo, hi) of the orbitals / targets rank `rank` owns: contiguous blocks, sizes differing by at most one."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allgather_orbitals(phi_local, n_total: int, wire: str = "fp64"):
    """All ranks' orbital blocks -> the full set on every rank (identity when torch.distributed is not initialised).
    wire = "fp32": single precision on the wire, converted back to fp64 on arrival ("negligible changes
    in the accuracy" -- relative error <= 2^-24 per component; NOT used for parity-checked runs)."""
    import torch
    dist = dist_or_none()
    if dist is None:
        return phi_local
    world, rank = dist.get_world_size(), dist.get_rank()
    counts = [shard_range(n_total, world, r) for r in range(world)]
    assert phi_local.shape[0] == counts[rank][1] - counts[rank][0], "local block does not match shard_range"
    send = phi_local.to(torch.complex64) if wire == "fp32" else phi_local
    # (re, im) pairs as real numbers on the wire: every backend moves floats
    send_r = torch.view_as_real(send.contiguous())
    # blocks differ by at most one orbital: every rank sends max-size blocks (collectives want equal sizes)
    cmax = max(hi - lo for lo, hi in counts)
    pad = torch.zeros((cmax,) + tuple(send_r.shape[1:]), dtype=send_r.dtype, device=phi_local.device)
    pad[:send_r.shape[0]] = send_r
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    full_r = torch.cat([parts[r][:hi - lo] for r, (lo, hi) in enumerate(counts)])
    full = torch.view_as_complex(full_r.contiguous())
    return full.to(torch.complex128) if wire == "fp32" else full


def sharded_apply(plan, phi_local, n_total: int, wire: str = "fp64"):
    """(V_X[Phi] phi_j) for the targets this rank owns: all-gather Phi, then one j-block apply.  Returns
    (out_local, (lo, hi))."""
    dist = dist_or_none()
    world, rank = (dist.get_world_size(), dist.get_rank()) if dist is not None else (1, 0)
    lo, hi = shard_range(n_total, world, rank)
    phi = allgather_orbitals(phi_local, n_total, wire)
    return plan.apply(phi, None, self_offset=lo, n_targets=hi - lo), (lo, hi)
