"""One-process-per-GPU sharding of the stream id space.

Streams are independent units, so the path shards with NO data-path
collective: rank p of P owns a contiguous block of global stream ids and creates its
handle with rng_create_shard(kind, n_total, first, n_local, seed).  Seeding is random
access in the global stream id (splitmix64 index, Philox key, LCG jump-ahead), so every
rank's rows are bit-identical to the same rows of a single-GPU run.  Host logic only.
"""
from __future__ import annotations


def shard_range(rank: int, world: int, n_total: int, granule: int = 1) -> tuple[int, int]:
    """-> (first, n_local): contiguous, covering [0, n_total) exactly once over ranks,
    block sizes differing by at most one granule (granule = 32 for RNG_XS1024W, whose
    streams come in whole 32-word instances)."""
    if not (0 <= rank < world) or n_total < 0 or granule < 1 or n_total % granule:
        raise ValueError("shard_range: bad arguments")
    units = n_total // granule
    base, rem = divmod(units, world)
    first_u = rank * base + min(rank, rem)
    n_u = base + (1 if rank < rem else 0)
    return first_u * granule, n_u * granule


def weak_scaling_shard(rank: int, world: int, n_per_gpu: int) -> tuple[int, int, int]:
    """bench.py's weak-scaling layout: every rank gets n_per_gpu streams of a global
    space of world*n_per_gpu.  -> (n_total, first, n_local)"""
    if not (0 <= rank < world) or n_per_gpu < 1:
        raise ValueError("weak_scaling_shard: bad arguments")
    return world * n_per_gpu, rank * n_per_gpu, n_per_gpu
