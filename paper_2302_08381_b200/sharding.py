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


def compute_sharded(xyz_host, l_max: int, normalized: bool = True, gradients: bool = False,
                    hessians: bool = False, devices=None):
    """N-sharded forward over every visible GPU from ONE process: shard r of ``xyz_host`` ([n,3]
    host tensor, pinned for full PCIe rate) goes to device r on a stream of its own, the forward
    kernel runs there, and the outputs stay on that GPU (no collective: P:118).  Returns
    ``[(start, stop, sph, dsph, ddsph), ...]`` per device, all work enqueued and NOT synchronised:
    the caller synchronises the devices it reads from.  Marshalling only; the arithmetic is the
    library's (``compute``)."""
    import torch

    from . import compute

    if devices is None:
        devices = list(range(torch.cuda.device_count()))
    if not devices:
        raise RuntimeError("compute_sharded: no CUDA device (there is no CPU fallback)")
    n, out = xyz_host.shape[0], []
    for r, dev in enumerate(devices):
        a, b = shard_range(n, r, len(devices))
        with torch.cuda.device(dev):
            stream = torch.cuda.Stream()
            with torch.cuda.stream(stream):
                x = xyz_host[a:b].to(f"cuda:{dev}", non_blocking=True)
                sph, dsph, ddsph = compute(x, l_max, normalized, gradients, hessians)
        out.append((a, b, sph, dsph, ddsph))
    return out
