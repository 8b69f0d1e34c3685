"""Multi-GPU plumbing of bench.py: one process per GPU, independent rollout groups per rank.

The attention hot path of one rollout group has no cross-GPU exchange (whole groups
on different GPUs are independent), so ranks shard GROUPS, never a group: weak scaling, no data-path
collective.  The only collectives are the timing ones -- a barrier around the timed region and a MAX
over ranks of the device time.  Works with the `nccl` backend on GPUs and with `gloo` on CPU (tests).
"""
from __future__ import annotations

import copy

import torch
import torch.distributed as dist

RANK_SEED_STRIDE = 100000


def rank_shape(shape, rank: int):
    """Rank r draws its own rollout group: same shapes, seed shifted by r * RANK_SEED_STRIDE."""
    s = copy.deepcopy(shape)
    s.seed = shape.seed + RANK_SEED_STRIDE * int(rank)
    return s


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a per-rank scalar (the timed milliseconds); identity when not distributed."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, ms_max: float, world: int) -> float:
    """Whole-job throughput: units all ranks processed / the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)
