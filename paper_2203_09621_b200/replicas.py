"""Replicas-only multi-GPU plumbing: N independent problems, one per rank.

The path does not shard (north_star: one GPU, no collectives), so the only cross-rank traffic is the
bench contract's barrier and the final max / sum of a few scalars.  These helpers are backend-agnostic
(`nccl` on the GPU box, `gloo` in the CPU tests) and hold no arithmetic of the method.
"""
from __future__ import annotations

import os

BASE_SEED = 20220309


def env_ranks():
    """(rank, local_rank, world_size) from the torchrun environment (1 process when unset)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def replica_seed(config_index: int, rank: int):
    """Rank 0 solves the configuration's own seeded problem (None = the config's seed); rank r > 0 a
    different member of the same family, so that replicas do not share a matrix."""
    return None if rank == 0 else BASE_SEED + int(config_index) + 1000 * int(rank)


def _reduce(x: float, op_name: str, device):
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(x: float, device="cpu") -> float:
    return _reduce(x, "MAX", device)


def sum_over_ranks(x: float, device="cpu") -> float:
    return _reduce(x, "SUM", device)


def whole_job_rate(units_this_rank: float, ms_this_rank: float, device="cpu") -> float:
    """Bench contract: units all ranks processed / the slowest rank's time (units per second)."""
    return sum_over_ranks(units_this_rank, device) / (max_over_ranks(ms_this_rank, device) * 1e-3)
