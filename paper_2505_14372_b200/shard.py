"""Position sharding across GPUs: host-side plumbing only, no arithmetic of the method.

Given the object and the probe, probe positions are independent units, so the path shards over
positions with object / probe replicated.  The one exchange step per batch is a sum of the quantities every
rank accumulates over ITS positions: object gradient, probe gradient, illumination map, loss.  Per-position
outputs (position gradients, per-position losses, step terms) stay with the rank that owns the rows.
`torch.distributed` (NCCL on GPUs, gloo in the CPU tests) does the reduction.
"""
from __future__ import annotations

from typing import Iterable, Optional

import numpy as np


def shard_rows(n_pos: int, rank: int, world: int) -> np.ndarray:
    """Rows of positions / intensities owned by `rank`: contiguous, balanced to within one row, int32."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    base, extra = divmod(n_pos, world)
    lo = rank * base + min(rank, extra)
    return np.arange(lo, lo + base + (1 if rank < extra else 0), dtype=np.int32)


def shard_batches(batches: Iterable[np.ndarray], rank: int, world: int):
    """Split every mini-batch (PAPER.md:55 'group') across ranks, keeping the batch order: rank r gets the
    r-th balanced slice of each batch, so all ranks step through the same sequence of batches."""
    out = []
    for b in batches:
        b = np.asarray(b, np.int32)
        out.append(b[shard_rows(b.size, rank, world)])
    return out


def allreduce_sums(dist, *tensors, group=None) -> None:
    """In-place sum over ranks of every given tensor (None entries are skipped).  Complex tensors are reduced
    through their real view.  `dist` is torch.distributed (already initialised) or None for a single process."""
    if dist is None:
        return
    import torch
    for t in tensors:
        if t is None:
            continue
        dist.all_reduce(torch.view_as_real(t) if t.is_complex() else t, op=dist.ReduceOp.SUM, group=group)
