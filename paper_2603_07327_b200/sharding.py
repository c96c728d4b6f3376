"""Host-side partition of histories across ranks (bench.py --gpus N).

The path is embarrassingly parallel over histories and every draw is a pure function of (seed,
history, stream, index) [R1], so ranks take disjoint history ranges and never exchange data during
transport or digitizing; ranges are aligned to time slices [R16] so no coincidence window straddles
two ranks.  north_star keeps the product single-GPU; this is only the bench's weak-scaling harness.
"""
from __future__ import annotations

from typing import Tuple


def history_range(rank: int, world_size: int, pairs_per_rank: int) -> Tuple[int, int]:
    """Weak scaling: rank r simulates [r * pairs_per_rank, (r + 1) * pairs_per_rank)."""
    if not (0 <= rank < world_size) or pairs_per_rank < 0:
        raise ValueError("bad rank / world_size / pairs_per_rank")
    return rank * pairs_per_rank, pairs_per_rank


def total_pairs(world_size: int, pairs_per_rank: int) -> int:
    return world_size * pairs_per_rank


def max_over_ranks(value: float) -> float:
    """Max of a scalar over all ranks (the job's time is the slowest rank's); identity without a group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
