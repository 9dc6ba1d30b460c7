"""Multi-GPU plumbing for the source update: cells are independent, so N
ranks simply own N disjoint cell ranges and NO collective touches the data path.  Weak scaling
(bench.py): rank r generates and updates cells [r*n, (r+1)*n) of the seeded workload.  The only
cross-rank operations are a barrier and a MAX/SUM all-reduce of timings and diagnostic counters.
"""
from __future__ import annotations


def rank_cell_range(cells_per_rank: int, rank: int) -> tuple[int, int]:
    """(first cell, count) of the seeded workload owned by `rank` under weak scaling."""
    if cells_per_rank < 0 or rank < 0:
        raise ValueError("cells_per_rank and rank must be non-negative")
    return rank * cells_per_rank, cells_per_rank


def split_cells(total_cells: int, world: int) -> list[tuple[int, int]]:
    """Strong-scaling split of `total_cells` into `world` contiguous ranges whose sizes differ by at most 1."""
    if world < 1 or total_cells < 0:
        raise ValueError("world must be >= 1 and total_cells >= 0")
    base, rem = divmod(total_cells, world)
    out, start = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((start, n))
        start += n
    return out


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """MAX all-reduce of a scalar (timings are reported as the slowest rank's)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(values, dist=None, device="cpu"):
    """SUM all-reduce of a list of integer counters (diagnostics only)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [int(v) for v in values]
    import torch

    t = torch.tensor([int(v) for v in values], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [int(v) for v in t.tolist()]
