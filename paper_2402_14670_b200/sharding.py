"""Multi-GPU plumbing: the path shards by events with NO data-path collective.

Events are independent: each rank runs the whole hot path on its own events.
``torch.distributed`` is used only for the barrier and for reducing the timing / counts
(NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import List, Tuple

import numpy as np


def event_ranges(seed_offsets: np.ndarray, world_size: int) -> List[Tuple[int, int]]:
    """Contiguous event ranges, one per rank, balanced by seed count (the unit of work)."""
    so = np.asarray(seed_offsets).astype(np.int64)
    n_ev = so.shape[0] - 1
    cuts = [0]
    for r in range(1, world_size):
        target = (so[-1] * r) // world_size
        c = int(np.searchsorted(so, target, side="left"))
        cuts.append(min(max(c, cuts[-1]), n_ev))
    cuts.append(n_ev)
    return [(cuts[r], cuts[r + 1]) for r in range(world_size)]


def dist_env() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process if unset)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def reduce_job(local_ms: float, local_counts, device=None):
    """Whole-job numbers: max over ranks of the device time, sum over ranks of the unit counts."""
    import torch
    import torch.distributed as dist
    counts = [float(c) for c in local_counts]
    if not (dist.is_available() and dist.is_initialized()):
        return local_ms, counts
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    c = torch.tensor(counts, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(v) for v in c.tolist()]
