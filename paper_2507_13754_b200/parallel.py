"""Host logic for runs on more than one GPU (one process per GPU, torch.distributed).

A single Born-series solve does not shard ("replicas only"); what shards is the
frequency batch -- independent plans, no data-path collective.  The only communication is the
bench contract's reduction of timings (MAX over ranks) and counts (SUM over ranks).
"""
from __future__ import annotations


def shard_frequencies(nfreq: int, rank: int, world: int) -> list:
    """Contiguous, balanced block of frequency indices owned by `rank` (may be empty)."""
    if not (0 <= rank < world) or nfreq < 0:
        raise ValueError("bad rank/world/nfreq")
    base, extra = divmod(nfreq, world)
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def reduce_timing(dist, device, times, counts):
    """MAX over ranks of `times` (list of floats) and SUM over ranks of `counts` (list of numbers).

    `dist` is torch.distributed (already initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(t) for t in times], [float(c) for c in counts]
    import torch
    t = torch.tensor([float(v) for v in times], dtype=torch.float64, device=device)
    c = torch.tensor([float(v) for v in counts], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist(), c.tolist()
