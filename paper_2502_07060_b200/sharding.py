"""Batch sharding for N GPUs: points are independent, so
rank r of `world` owns a contiguous slice of the seeded workload and no data-path collective
exists.  Host logic only; used by bench.py and covered by tests/test_sharding.py (gloo)."""
from __future__ import annotations


def weak_slice(rank: int, world: int, batch_per_rank: int) -> tuple[int, int]:
    """weak scaling: every rank processes `batch_per_rank` points; rank r owns global points
    [r*batch_per_rank, (r+1)*batch_per_rank) of a workload of world*batch_per_rank points"""
    if not (0 <= rank < world) or batch_per_rank < 0:
        raise ValueError("bad (rank, world, batch)")
    return rank * batch_per_rank, batch_per_rank


def strong_slice(rank: int, world: int, total: int) -> tuple[int, int]:
    """strong scaling: `total` points cut into `world` contiguous slices whose sizes differ by
    at most one (the first total % world ranks get the extra point); returns (start, count)"""
    if not (0 <= rank < world) or total < 0:
        raise ValueError("bad (rank, world, total)")
    q, r = divmod(total, world)
    start = rank * q + min(rank, r)
    return start, q + (1 if rank < r else 0)
