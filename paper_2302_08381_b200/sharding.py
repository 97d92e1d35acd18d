"""Multi-GPU: the path shards over points with no communication ("trivially parallelized
over the sample index").  One process per GPU; rank r owns a contiguous range of the N points and
the matching rows of sph / dsph / ddsph / grad_xyz stay on its GPU.  No collective is on the data
path; torch.distributed is used only for the barrier and the max-over-ranks timing in bench.py.
"""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int, align: int = 32) -> tuple[int, int]:
    """[start, stop) of rank's points: contiguous, disjoint, covering [0,n); interior boundaries
    are multiples of ``align`` (a 32-point tile never straddles two GPUs)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    tiles = (n + align - 1) // align
    base, extra = divmod(tiles, world)
    t0 = rank * base + min(rank, extra)
    t1 = t0 + base + (1 if rank < extra else 0)
    return min(t0 * align, n), min(t1 * align, n)
