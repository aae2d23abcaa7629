"""Host-side logic of the multi-GPU launch: one process per GPU, one independent
cluster per rank, no data-path collective.  The only exchanges are the timing reductions below, so this
module runs unchanged on the gloo backend (tests/test_multi_rank.py, world_size 2 on CPU).
"""
from __future__ import annotations

from . import workloads


def rank_config(config_id, rank, n=None):
    """Workload of one rank: BASELINE.json config `config_id` with the recipe's seed advanced by 100 per
    rank (rank 0 is the single-GPU workload itself), same parameters on every rank (weak scaling)."""
    return workloads.config(config_id, n=n, seed_offset=100 * rank)


def aggregate(dist, local_units, local_ms, device="cpu"):
    """Whole-job figures from per-rank ones: units summed over ranks, time = the slowest rank's
    (`dist` = torch.distributed or None for a single process).  Returns (total_units, max_ms)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return int(local_units), float(local_ms)
    import torch

    t = torch.tensor([float(local_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([int(local_units)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return int(u.item()), float(t.item())


def throughput(total_units, max_ms):
    """units per second of the whole job."""
    return total_units / (max_ms * 1e-3)


# ---- one evaluation sharded over the ranks (include/p3t.h p3t_set_shard) ---------------------
# Every rank holds all particles and the same tree and walks every world-th i-group; a particle's acceleration,
# potential and neighbour list are produced by exactly one rank and are zero / empty on the others.

def merge_forces(parts):
    """acc [n,3] / pot [n] arrays of all ranks -> the full result (a sum with zeros: exact)."""
    out = parts[0].copy()
    for p in parts[1:]:
        out += p
    return out


def merge_csr(parts, n):
    """[(offset[n+1], nbr[total_r]) per rank] -> (offset[n+1] uint64, nbr[total] uint32) of all particles."""
    import numpy as np

    counts = [np.diff(off.astype(np.int64)) for off, _ in parts]
    total = np.zeros(n, dtype=np.int64)
    for c in counts:
        total += c
    offset = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(total, out=offset[1:])
    nbr = np.empty(int(offset[-1]), dtype=np.uint32)
    for (off, lst), c in zip(parts, counts):
        t = int(c.sum())
        if t == 0:
            continue
        start_local = np.repeat(off[:-1].astype(np.int64), c)
        start_global = np.repeat(offset[:-1], c)
        nbr[start_global + (np.arange(t, dtype=np.int64) - start_local)] = lst[:t]
    return offset.astype(np.uint64), nbr


def allreduce_forces(dist, acc, pot):
    """In-place sum over ranks of the torch tensors acc, pot (device tensors with NCCL, CPU tensors with gloo)."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(acc, op=dist.ReduceOp.SUM)
        dist.all_reduce(pot, op=dist.ReduceOp.SUM)
    return acc, pot


def allgather_csr(dist, offset, nbr, n):
    """Neighbour lists of all ranks on every rank (numpy in, numpy out)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return offset, nbr
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, (offset, nbr))
    return merge_csr(parts, n)
