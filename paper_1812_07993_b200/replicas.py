"""Multi-GPU bookkeeping: independent replicas, one per rank, no data-path collective.

torch.distributed is used only to line the ranks up (barrier) and to combine their timings: the job's
throughput is the units all ranks processed divided by the slowest rank's device time.
"""
from __future__ import annotations

import os

from . import inputs


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def replica_seed(base_seed: int, rank: int) -> int:
    """Distinct, reproducible seed of rank's replica (rank 0 keeps the config's own seed)."""
    return base_seed + 7919 * rank


def replica_config(rank: int):
    """BASELINE.json configs[2] for this rank's replica."""
    return inputs.config2(seed=replica_seed(inputs.BASE_SEED + 2, rank))


def _reduce(x: float, op, device):
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(x: float, device="cpu") -> float:
    import torch.distributed as dist

    return _reduce(x, dist.ReduceOp.MAX, device)


def sum_over_ranks(x: float, device="cpu") -> float:
    import torch.distributed as dist

    return _reduce(x, dist.ReduceOp.SUM, device)


def job_throughput(units_this_rank: float, seconds_this_rank: float, device="cpu"):
    """(whole-job units per second, slowest rank's seconds): sum of units / max of times."""
    t = max_over_ranks(seconds_this_rank, device)
    return sum_over_ranks(units_this_rank, device) / t, t
