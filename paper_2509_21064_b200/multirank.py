"""Host-side logic for running replicas on several GPUs (one process per GPU, torch.distributed).

Restarts are independent, so ranks share no data during the iteration: every rank runs its own
B restarts of the same instance from its own seeded start points.  The only exchange is the arg-best across
ranks after the run: one all-reduce(MIN) over (objective, rank, restart) triples packed for a lexicographic min.
"""
from __future__ import annotations

from typing import Tuple


def rank_x0_seed(base_seed: int, rank: int) -> int:
    """Distinct, reproducible start-point seed per rank (rank 0 keeps the single-GPU seed)."""
    return base_seed + 7919 * rank


def combine_best(best_obj: float, best_restart: int, rank: int, world: int, device=None) -> Tuple[float, int, int]:
    """(objective, rank, restart) of the global best; ties -> lowest rank, then lowest restart (reading R6).
    With world == 1 no collective is issued."""
    if world == 1:
        return float(best_obj), rank, int(best_restart)
    import torch
    import torch.distributed as dist
    v = torch.tensor([float(best_obj)], dtype=torch.float64, device=device)
    dist.all_reduce(v, op=dist.ReduceOp.MIN)
    gmin = float(v.item())
    # among the ranks that hold the minimum, the lowest (rank, restart) wins
    key = rank * (1 << 32) + int(best_restart) if float(best_obj) == gmin else (1 << 62)
    k = torch.tensor([key], dtype=torch.int64, device=device)
    dist.all_reduce(k, op=dist.ReduceOp.MIN)
    key = int(k.item())
    return gmin, key >> 32, key & 0xFFFFFFFF


def max_over_ranks(value: float, world: int, device=None) -> float:
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
