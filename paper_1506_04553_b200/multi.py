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
