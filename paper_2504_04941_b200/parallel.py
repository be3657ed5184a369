"""Multi-GPU plumbing: cells are independent, so the step shards with no data-path
collective.  One process per GPU; each rank integrates its own block-cyclic share of the cells; the only
collectives are the reductions of the six work counters and of the elapsed time (max over ranks).

Nothing here touches CUDA: the same functions run under the ``gloo`` backend in the CPU tests.
"""
from __future__ import annotations

from typing import Dict, Optional

import numpy as np


def shard_indices(n_cells: int, rank: int, world: int, block: int = 4096) -> np.ndarray:
    """Block-cyclic share of rank: blocks b with b % world == rank (stiff cells cluster in space --
    PAPER.md:507 -- so contiguous slabs would balance badly).  Disjoint over ranks, union = all cells."""
    if not (0 <= rank < world) or block <= 0 or n_cells < 0:
        raise ValueError("bad shard arguments")
    n_blocks = (n_cells + block - 1) // block
    mine = np.arange(rank, n_blocks, world, dtype=np.int64)
    if mine.size == 0:
        return np.zeros(0, np.int64)
    idx = (mine[:, None] * block + np.arange(block, dtype=np.int64)[None, :]).ravel()
    return idx[idx < n_cells]


def shard_cells(cells, rank: int, world: int, block: int = 4096):
    """The rank's share of a ``workloads.Cells`` (copies)."""
    return cells.take(shard_indices(cells.n_cells, rank, world, block))


def allreduce_stats(stats: Dict[str, int], group=None) -> Dict[str, int]:
    """Sum the work counters over ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return dict(stats)
    keys = sorted(stats)
    t = torch.tensor([int(stats[k]) for k in keys], dtype=torch.int64)
    if dist.get_backend(group) == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return {k: int(v) for k, v in zip(keys, t.cpu().tolist())}


def max_over_ranks(value: float, group=None) -> float:
    """Elapsed time of the slowest rank (device-measured milliseconds in, the maximum out)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64)
    if dist.get_backend(group) == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sum_over_ranks(value: float, group=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64)
    if dist.get_backend(group) == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t.item())
