"""Multi-GPU plumbing for independent particles ("trajectories are
independent ... trivially parallelized over CPUs or GPUs").

The path shards by particle with NO data-path collective: every rank holds the (<= 0.5 MB) field tables and
traces its own slice with the same kernel.  What crosses ranks is bookkeeping only: the timing reduction of
the benchmark (max over ranks), the attempt counters (sum) and, when a caller wants one array back, a gather
of the per-particle results.  ``torch.distributed`` carries it (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import numpy as np


def shard_indices(n_total: int, rank: int, world: int) -> np.ndarray:
    """Round-robin slice of one ensemble: particle i belongs to rank i mod world.  Round-robin (rather than
    contiguous blocks) spreads any ordering of the initial conditions -- and with it the strongly
    divergent step counts -- evenly over the ranks."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    return np.arange(rank, n_total, world, dtype=np.int64)


def unshard(parts, n_total: int) -> np.ndarray:
    """Inverse of ``shard_indices``: parts[r] holds the rows of rank r (last axis = particles)."""
    world = len(parts)
    first = np.asarray(parts[0])
    out = np.empty(first.shape[:-1] + (n_total,), dtype=first.dtype)
    for r, p in enumerate(parts):
        out[..., r::world] = np.asarray(p)
    return out


def reduce_timing(elapsed_ms: float, attempts: int, device=None):
    """(max over ranks of elapsed_ms, sum over ranks of attempts).  Without an initialised process group
    this is the identity."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(elapsed_ms), int(attempts)
    dev = device if device is not None else "cpu"
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=dev)
    a = torch.tensor([int(attempts)], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(a, op=dist.ReduceOp.SUM)
    return float(t.item()), int(a.item())


def gather_to_rank0(local: np.ndarray, n_total: int):
    """Gather round-robin shards (last axis = particles) of a result array onto rank 0, in ensemble order.
    Returns the full array on rank 0 and None elsewhere."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return np.asarray(local)
    world, rank = dist.get_world_size(), dist.get_rank()
    parts = [None] * world if rank == 0 else None
    dist.gather_object(np.asarray(local), parts, dst=0)
    return unshard(parts, n_total) if rank == 0 else None


def loss_fraction_curve(t_out: np.ndarray, status: np.ndarray, t_grid: np.ndarray, lost_code: int = 1):
    """Cumulative lost fraction at the times of ``t_grid`` from per-particle loss times (config 1's
    output, BASELINE.json: "loss fraction vs time and per-particle loss times")."""
    lost_t = np.sort(np.asarray(t_out)[np.asarray(status) == lost_code])
    return np.searchsorted(lost_t, np.asarray(t_grid), side="right") / float(len(t_out))
