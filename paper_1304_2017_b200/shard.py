"""Multi-GPU sharding of the path: transducers (rows of H) are
partitioned across ranks, the volume is replicated.  H needs no exchange (every rank owns its rows of
y); H^T produces one full-size partial volume per rank, summed by ONE all-reduce -- the paper's own
backward split by rings (Algs. 10-11) with the CPU-side sum replaced by NCCL.

Host-side logic only (no arithmetic of the method); covered on CPU with gloo in tests/test_shard.py.
"""
from __future__ import annotations

import numpy as np


def shard_range(n: int, rank: int, world: int) -> tuple:
    """Contiguous block partition of range(n): sizes differ by at most one, every index owned once."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_transducers(trans_xyz: np.ndarray, rank: int, world: int) -> np.ndarray:
    """Strong-scaling shard: this rank's rows of H."""
    lo, hi = shard_range(trans_xyz.shape[0], rank, world)
    return np.ascontiguousarray(trans_xyz[lo:hi])


def weak_replica_transducers(trans_xyz: np.ndarray, rank: int, world: int, n_views: int) -> np.ndarray:
    """Weak-scaling shard used by bench.py: rank r holds the same array rotated about z by
    r/world of one view step, i.e. the N ranks together form an N-times denser view sampling."""
    ang = 2.0 * np.pi / n_views * (rank / world)
    c, s = np.cos(ang), np.sin(ang)
    rot = np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])
    return np.ascontiguousarray(trans_xyz @ rot.T)


def allreduce_volume(x, group=None):
    """Sum the per-rank partial volumes of H^T in place (the path's one exchange step)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(x, op=dist.ReduceOp.SUM, group=group)
    return x
