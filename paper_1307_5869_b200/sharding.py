"""Multi-GPU plumbing: shard a block-split family by stream index, reduce timings over ranks.

Streams are independent and stream s's start is a closed-form function of (seed, s, block_len)
(PAPER.md:277), so each rank initialises and fills its own contiguous range of streams; there is no
exchange step on the data path.  Only ``torch.distributed`` plumbing lives here.
"""
from __future__ import annotations


def shard_streams(total_streams: int, rank: int, world: int) -> tuple[int, int]:
    """Strong split of ``total_streams`` columns: -> (first_stream, n_streams) of ``rank``.
    Contiguous ranges, sizes differ by at most one, earlier ranks take the larger ones."""
    if not (0 <= rank < world) or total_streams < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(total_streams, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def weak_shard(streams_per_rank: int, rank: int) -> tuple[int, int]:
    """Weak scaling (bench.py --gpus N): every rank holds ``streams_per_rank`` streams of ONE global
    family of world * streams_per_rank streams: -> (first_stream, n_streams)."""
    return rank * streams_per_rank, streams_per_rank


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar timing when a process group is up, else the value itself."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
