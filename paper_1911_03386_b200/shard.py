"""Multi-GPU layout of an ensemble (the paper ran independent
batches on its two GPUs).  Members are independent, so the path shards by member with NO
data-path collective: rank r owns a contiguous block of members and steps it alone.  The
only exchange is the tiny per-member series gathered once after the run (the ensemble
statistics of eq.(41), need every member's beta)."""
from __future__ import annotations


def member_range(total_members: int, rank: int, world: int):
    """Contiguous block [lo, hi) of members owned by `rank` (sizes differ by at most one)."""
    assert 0 <= rank < world and total_members >= 0
    base, extra = divmod(total_members, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def gather_series(local_series, total_members: int, group=None):
    """all_gather of series[samples][local_members][4] into [samples][total_members][4] (torch tensors,
    any backend: nccl on GPUs, gloo in the CPU tests).  Blocks are padded to the largest shard."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    sizes = [member_range(total_members, r, world) for r in range(world)]
    width = max(hi - lo for lo, hi in sizes)
    S = local_series.shape[0]
    pad = torch.zeros((S, width, 4), dtype=local_series.dtype, device=local_series.device)
    pad[:, : local_series.shape[1]] = local_series
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = torch.empty((S, total_members, 4), dtype=local_series.dtype, device=local_series.device)
    for (lo, hi), p in zip(sizes, parts):
        out[:, lo:hi] = p[:, : hi - lo]
    assert sizes[rank][1] - sizes[rank][0] == local_series.shape[1]
    return out


def max_over_ranks(seconds: float, device=None, group=None) -> float:
    """Device-timed duration of the slowest rank (the bench contract's max-over-ranks)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return seconds
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
