"""Multi-GPU host logic: the path has no exchange step, so N ranks run N replicas of the tables
and disjoint windows of the request stream (weak scaling).  The only cross-rank operation is the MAX of the
per-rank device time that bench.py reports.  No method arithmetic here; torch.distributed only."""
from __future__ import annotations


def rank_window(rank: int, world: int, n_per_rank: int) -> tuple[int, int]:
    """[start, stop) of the request stream that `rank` of `world` processes: consecutive, disjoint, equal-sized."""
    if not (0 <= rank < world) or n_per_rank < 0:
        raise ValueError("bad rank/world/n")
    return rank * n_per_rank, (rank + 1) * n_per_rank


def max_over_ranks(value: float, device=None) -> float:
    """MAX over all ranks of a host float (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """SUM over all ranks of a host float (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
