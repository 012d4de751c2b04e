"""Multi-GPU plumbing around liblra: one process per GPU, visibilities partitioned by contiguous
row (time) ranges, every rank grids its rows into a private full grid, one all-reduce combines the grids and the sums
of weights ("the outputs are combined by accumulation"; partitions by time and frequency).
Degridding needs no collective once every rank holds the model grid.  torch.distributed only: NCCL on GPUs, gloo in
the CPU tests.  No arithmetic of the method lives here."""
from __future__ import annotations

from typing import Tuple


def row_range(nrow: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [lo, hi) row range of `rank`: sizes differ by at most one row, earlier ranks get the longer ones."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank / world")
    base, extra = divmod(nrow, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def reduce_grid(grid, sumwt=None, group=None):
    """In-place sum over ranks of the complex grid [nterms, ncorr, ny, nx] and of sumwt (the data-path exchange step of
    gridding).  Returns (grid, sumwt)."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(torch.view_as_real(grid), group=group)
        if sumwt is not None:
            dist.all_reduce(sumwt, group=group)
    return grid, sumwt


def broadcast_model(grid, src: int = 0, group=None):
    """Gives every rank the model grid before degridding (once per major cycle)."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.broadcast(torch.view_as_real(grid), src=src, group=group)
    return grid
