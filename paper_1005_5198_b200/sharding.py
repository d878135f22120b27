"""Multi-GPU sharding of one map: rays are independent, so the n1 x n2 ray
grid is cut into row bands, one per rank (the paper's own runs split ray batches over 2 or
4 GPUs).  Every rank holds all lenses (<= 324 KB) and a private uint32
map; the one exchange step is a sum of the maps (NCCL all-reduce over NVLink on GPUs, gloo
in the CPU tests).  Host logic only -- no arithmetic of the method.
"""
from __future__ import annotations


def row_band(n2: int, rank: int, world: int, align: int = 1):
    """Rows [j0, j1) of rank `rank`: bands are contiguous, disjoint, cover [0, n2), differ
    by at most `align` rows in height and start on multiples of `align` (the kernel's tile
    height, so that no tile is split between two ranks)."""
    if world < 1 or not (0 <= rank < world) or n2 < 0 or align < 1:
        raise ValueError("row_band: bad arguments")
    units = -(-n2 // align)  # tile rows, the last may be ragged
    lo = (units * rank) // world
    hi = (units * (rank + 1)) // world
    return min(lo * align, n2), min(hi * align, n2)


def allreduce_map(counts, group=None):
    """Sum the per-rank count maps in place on every rank.  `counts` is a torch int32 tensor
    viewing the uint32 map (two's-complement addition is the same bit pattern)."""
    import torch
    import torch.distributed as dist
    assert counts.dtype == torch.int32
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
    return counts
