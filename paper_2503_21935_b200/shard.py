"""Event sharding across ranks: events are independent ("event-level data parallelism"), so
rank r of N takes the contiguous range [r * per_rank, (r+1) * per_rank) of the seeded event stream; there is no
exchange step and no data-path collective ("replicas only").  Only the timing is reduced
(max over ranks)."""
from __future__ import annotations


def rank_range(per_rank: int, rank: int, world: int) -> tuple[int, int]:
    """[start, stop) of the global event stream owned by `rank` (weak scaling: per_rank fixed as world grows)."""
    if not (0 <= rank < world) or per_rank < 0:
        raise ValueError("bad rank/world/per_rank")
    return rank * per_rank, (rank + 1) * per_rank


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """max of a host float over all ranks of the default process group (identity without a group)."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
