"""Multi-GPU plumbing of bench.py: the path has no exchange step (replicas only), so ranks only agree
on the step time (max over ranks) after the timed region.  Kept here so that the N>1 logic can be tested on CPU with gloo."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def world():
    return int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))


def rank_seed(rank: int, base_seed: int = 0) -> int:
    """Every rank renders its own scene of the same recipe."""
    return base_seed + rank


def max_over_ranks(values, device="cpu"):
    """values: list of floats measured on this rank -> list of the maxima over all ranks (identity for one process)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_throughput(units_per_rank: float, ms_step_max: float, world_size: int) -> float:
    """whole-job units per second: every rank processes units_per_rank in the slowest rank's step time."""
    return world_size * units_per_rank / (ms_step_max * 1e-3)
