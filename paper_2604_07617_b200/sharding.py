"""Particle-sharded runs (particles are independent, Eq. 2 is a mean).

One seeded ensemble is split over the ranks by interleaved index (rank r takes particles r, r + N, r + 2N, ...:
loss time correlates with the birth radius, so contiguous blocks would be unevenly loaded), every rank builds
the same tables and traces its share with catapult_trace; the only exchange of the whole job is ONE all-reduce of
(sum g, sum g^2, n) -- 24 bytes -- from which every rank gets Eq. 2's estimate and its standard error.  There is
no data-path collective: nothing here touches the kernels.

Host-side plumbing only (torch.distributed: NCCL on GPUs, gloo in the CPU tests); none of the method's arithmetic.
"""
from __future__ import annotations

import math

import numpy as np


def shard_indices(n: int, rank: int, world: int) -> np.ndarray:
    """Indices of the ensemble's particles that rank `rank` of `world` traces: rank, rank + world, ..."""
    if not (0 <= rank < world):
        raise ValueError("rank must be in [0, world)")
    return np.arange(rank, n, world, dtype=np.int64)


def shard_columns(x0: np.ndarray, rank: int, world: int) -> np.ndarray:
    """The columns of a [4][n] initial-state array this rank traces (contiguous copy)."""
    return np.ascontiguousarray(x0[:, rank::world])


def gather_order(n: int, world: int) -> np.ndarray:
    """Position in the ensemble of every element of the rank-major concatenation of the shards:
    ensemble[gather_order] = concatenate(shards)."""
    return np.concatenate([shard_indices(n, r, world) for r in range(world)])


def reduce_estimate(sum_g: float, sum_g2: float, n: int, group=None, device=None):
    """All-reduces (sum g, sum g^2, n) over the ranks (one 24-byte collective) and returns Eq. 2's estimate:
    (mean, standard error sqrt((sum g^2 / n - mean^2) / (n - 1)), sum g, sum g^2, n), identical on every rank.
    For an indicator g the sums are integer counts below 2^53: the reduced count is exact whatever the order
    of the reduction.  Without an initialised process group (single rank) nothing is exchanged."""
    import torch
    import torch.distributed as dist

    v = torch.tensor([float(sum_g), float(sum_g2), float(n)], dtype=torch.float64, device=device or "cpu")
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(v, op=dist.ReduceOp.SUM, group=group)
    s, s2, nn = (float(t) for t in v.tolist())
    mean = s / nn if nn > 0 else 0.0
    var = (s2 / nn - mean * mean) / (nn - 1.0) if nn > 1 else 0.0
    return mean, math.sqrt(max(var, 0.0)), s, s2, int(round(nn))


def reduce_timing(seconds: float, counts, group=None, device=None):
    """Whole-job figures of a sharded run: the time is the MAX over ranks, every count the SUM over ranks."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1):
        return float(seconds), [float(c) for c in counts]
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device or "cpu")
    c = torch.tensor([float(v) for v in counts], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    dist.all_reduce(c, op=dist.ReduceOp.SUM, group=group)
    return float(t.item()), [float(v) for v in c.tolist()]
