"""Multi-GPU plumbing: "replicas only".

One reduction does not shard without a per-panel broadcast pipeline, and the largest config fits
one B200, so N GPUs run N independent matrices (the finite-field workflow of several primes /
several systems).  There is no data-path collective; torch.distributed is used only
for the barrier and the max-over-ranks timing that bench.py reports.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def replica_seed(base_seed: int, rank: int) -> int:
    """Each rank reduces its own matrix: same recipe, seed shifted by the rank."""
    return base_seed + 1000 * rank


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a host scalar (identity when not running under torch.distributed)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, seconds_max: float, world: int) -> float:
    """Whole-job throughput: all ranks' units divided by the slowest rank's time (weak scaling)."""
    return world * units_per_rank / seconds_max
