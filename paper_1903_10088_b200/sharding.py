"""Multi-GPU scheduling of independent slices: batch sharding, no data-path collective.

Slices of a stack are independent reconstructions (the paper reconstructs one slice at a time,
PAPER.md:156), so N GPUs = N processes that each own a contiguous block of slices and never exchange
image or sinogram data.  ``torch.distributed`` is used for exactly two things: a barrier around the
timed region and a max-reduction of the per-rank device time.  Works with the ``nccl`` backend on
GPUs and with ``gloo`` on CPU (tests).
"""
from __future__ import annotations

from typing import Tuple


def slice_range(rank: int, world_size: int, n_slices: int) -> Tuple[int, int]:
    """Contiguous block [lo, hi) of `n_slices` owned by `rank`; sizes differ by at most one, lower ranks
    take the remainder."""
    if world_size <= 0 or not (0 <= rank < world_size) or n_slices < 0:
        raise ValueError("bad rank/world_size/n_slices")
    base, rem = divmod(n_slices, world_size)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """Every rank gets the maximum of `value` (device time of the slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """Every rank gets the sum of `value` (units processed by the whole job)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
