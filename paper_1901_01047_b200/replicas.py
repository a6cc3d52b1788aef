"""Replicas-only multi-GPU plumbing.

Markov chains are independent, so N GPUs run N independent replicas of the
batched walker: rank r owns the walkers with seeds r*B .. r*B+B-1.  No data-path collective
exists; torch.distributed only carries the barrier, the max-over-ranks of the device time and the
sum of the work counters.  No CT-AUX arithmetic here.
"""
from __future__ import annotations

import numpy as np


def rank_seeds(rank: int, walkers_per_rank: int) -> np.ndarray:
    """Seeds of the walkers rank `rank` owns (walker w of the whole job uses seed w)."""
    first = rank * walkers_per_rank
    return np.arange(first, first + walkers_per_rank, dtype=np.uint64)


def aggregate(ms_local: float, counters_local, device="cpu"):
    """(max over ranks of the time, sum over ranks of each counter).  Works without an initialised
    process group (single replica)."""
    import torch
    import torch.distributed as dist
    counters_local = [float(c) for c in counters_local]
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), counters_local
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(counters_local, dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(x) for x in c.tolist()]
