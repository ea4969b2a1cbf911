"""Host-side helpers for running on several GPUs (one process per GPU, torch.distributed).

The search partitions with no data-path exchange:
  * by stack  -- every rank searches its own stack (one CCD per GPU); this is what bench.py does
                 for N > 1 ("weak" scaling);
  * by trajectory -- ranks share one stack and take disjoint slices of the trajectory bank; the
                 outputs (maps, candidate lists) of different trajectories are disjoint, so they
                 are simply concatenated in rank order.
Only a max-over-ranks reduction of the elapsed time crosses ranks.
"""
from __future__ import annotations

import dataclasses
from typing import Tuple


def shard_trajectories(n_traj: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced slice [lo, hi) of the trajectory bank for `rank` of `world`."""
    if not (0 <= rank < world) or n_traj < 0:
        raise ValueError("bad rank/world/n_traj")
    base, extra = divmod(n_traj, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def rank_config(cfg, rank: int):
    """The same recipe with a rank-specific seed (a different stack per GPU)."""
    return dataclasses.replace(cfg, idx=cfg.idx + 10 * rank) if rank else cfg


def aggregate_value(evals_per_rank: int, world: int, max_ms_per_step: float) -> float:
    """Whole-job evaluations per second: all ranks' work over the slowest rank's time."""
    return evals_per_rank * world / (max_ms_per_step * 1e-3)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a Python float over the default process group (no-op without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
