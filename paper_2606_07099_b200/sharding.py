"""Scenario sharding for more than one GPU (every scenario is an independent
diagonal block of the block-diagonal embedding, so the batch partitions with NO data-path collective).

One process per GPU; each rank builds the same template (sable_create on the same Y_bus) and solves a contiguous
range of scenarios.  torch.distributed is used only for plumbing around the path: a barrier, the max-over-ranks
time, the sum of converged counts and an optional gather of the result shards.
"""
from __future__ import annotations


def shard_range(batch: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced partition of range(batch): the first batch % world ranks get one extra scenario."""
    if world < 1 or not (0 <= rank < world) or batch < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(batch, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def reduce_job(local_seconds: float, local_converged: int, local_solves: int, device=None):
    """(max seconds over ranks, total converged, total solves).  No-op without an initialised process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local_seconds, local_converged, local_solves
    t = torch.tensor([local_seconds], dtype=torch.float64, device=device)
    c = torch.tensor([local_converged, local_solves], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), int(c[0].item()), int(c[1].item())


def gather_rows(local, batch: int, dst: int = 0):
    """Gather per-rank row shards (torch tensors, first dim = this rank's scenarios) into the global order on `dst`.
    Returns the full tensor on `dst`, None elsewhere."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(), dist.get_rank()
    sizes = [shard_range(batch, r, world) for r in range(world)]
    pad = max(hi - lo for lo, hi in sizes)
    buf = torch.zeros((pad,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    buf[: local.shape[0]] = local
    out = [torch.zeros_like(buf) for _ in range(world)] if rank == dst else None
    dist.gather(buf, out, dst=dst)
    if rank != dst:
        return None
    return torch.cat([out[r][: hi - lo] for r, (lo, hi) in enumerate(sizes)], dim=0)
