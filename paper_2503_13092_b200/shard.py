"""Multi-GPU sharding of the path: events are independent (P:149 one block per event, P:147 a farm of
independent GPUs), so rank r owns a contiguous range of events, runs the whole path on it with its own handle, and
there is NO collective on the data path.  The only exchange is an all-gather of three counters per rank, from which
every rank derives the global offsets of its tracks and vertices.  Host logic only; works on gloo and nccl.
"""
from __future__ import annotations


def event_range(rank: int, world_size: int, n_events: int) -> tuple[int, int]:
    """Contiguous, balanced split of [0, n_events): the first n_events % world_size ranks hold one extra event."""
    if not (0 <= rank < world_size) or n_events < 0:
        raise ValueError("bad rank / world_size / n_events")
    q, r = divmod(n_events, world_size)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def block_range(rank: int, blocks_per_rank: int) -> tuple[int, int]:
    """Weak scaling: rank r generates RNG blocks [r*B, (r+1)*B) of the config, i.e. its own distinct events."""
    return rank * blocks_per_rank, (rank + 1) * blocks_per_rank


def gather_counts(n_events: int, n_tracks: int, n_vertices: int, device=None):
    """All-gather (n_events, n_tracks, n_vertices) over the default process group.

    Returns (counts[world][3], my_offsets[3]) as python lists: my_offsets are the exclusive prefix sums, i.e. where
    this rank's events / tracks / vertices start in the global numbering."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        return [[n_events, n_tracks, n_vertices]], [0, 0, 0]
    world, rank = dist.get_world_size(), dist.get_rank()
    mine = torch.tensor([n_events, n_tracks, n_vertices], dtype=torch.int64, device=device)
    out = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(out, mine)
    counts = [t.tolist() for t in out]
    offs = [sum(c[k] for c in counts[:rank]) for k in range(3)]
    return counts, offs


def max_over_ranks(value: float, device=None) -> float:
    """Timing rule: a multi-GPU time is the maximum over ranks."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
