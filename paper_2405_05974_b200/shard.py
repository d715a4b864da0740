"""Data parallelism over cells (the only parallelism of this path: cells are independent).

No data-path collective exists: every rank creates its own `QssMech` (the tables are a few tens of KB) and evaluates a
contiguous range of cells.  The only communication is the timing reduction of bench.py (max over ranks).
"""
from __future__ import annotations


def cell_range(n_cells: int, rank: int, world: int, align: int = 32):
    """Contiguous [begin, end) of the cells owned by `rank`; boundaries are multiples of `align` (a slab of 32
    cells is the kernels' unit of work) except the last end, which is n_cells. Ranges tile [0, n_cells) exactly."""
    if world < 1 or not (0 <= rank < world) or n_cells < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, n_cells >= 0")
    slabs = (n_cells + align - 1) // align
    per, extra = divmod(slabs, world)
    b = rank * per + min(rank, extra)
    e = b + per + (1 if rank < extra else 0)
    return min(b * align, n_cells), min(e * align, n_cells)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """Max of a host float over all ranks (used for the timed region of bench.py); identity without a group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
