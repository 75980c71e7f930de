"""Multi-GPU host logic: the Sketch&Walk path shards only as independent replicas (one process per
GPU, each sequence owns its walk state R and its block lists), so there
is no data-path collective.  What ranks share is bookkeeping: distinct seeds per rank, the step time as
the maximum over ranks, and the whole-job throughput.  Works with any torch.distributed backend (NCCL on
GPUs, gloo in the CPU tests)."""
from __future__ import annotations

from typing import Optional

import torch


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of a rank's replica: rank 0 keeps the single-GPU seed, other ranks get disjoint streams."""
    return base_seed + 100003 * rank


def max_over_ranks(value: float, dist=None, device: Optional[torch.device] = None) -> float:
    """Step time of the job = slowest rank.  ``dist`` is torch.distributed (initialised) or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_throughput(units_per_rank: float, world: int, seconds: float) -> float:
    """Weak scaling: every rank processes ``units_per_rank`` units in the same (max-over-ranks) time."""
    return world * units_per_rank / seconds
