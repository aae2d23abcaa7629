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


def allreduce_shard(dist, ctx, rec=None):
    """The exchange of one sharded evaluation: ONE all-reduce (sum) of the records (a, phi, cost class + 1) of all
    particles (20 bytes per particle over NVLink with NCCL; `rec` may be a caller-owned [n, 5] float32 tensor), after
    which every rank holds the accelerations and potentials of all particles and hands the summed cost classes back to
    its context, so that the next sharded walk deals the groups out by predicted cost, the same way on every rank
    (include/p3t.h p3t_get_shard_record / p3t_put_shard_classes).  `ctx` needs get_shard_record(rec) and
    put_shard_classes(rec).  Returns (acc [n, 3], pot [n]) as views of the record."""
    rec = ctx.get_shard_record(rec)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(rec, op=dist.ReduceOp.SUM)
    ctx.put_shard_classes(rec)
    r = rec.view(-1, 5)
    return r[:, :3], r[:, 3]


def allgather_csr_tensors(dist, count, nbr):
    """Neighbour lists of all ranks on every rank, as tensors (NCCL with device tensors, gloo with CPU tensors; nothing
    is pickled).  count [n] int64 and nbr [total_r] int64/int32: this rank's list lengths (zero for the particles other
    ranks produced) and entries, lists in particle order.  Two collectives: an all-reduce of the lengths (every list has
    one owner, so the sum is the global length) and an all-gather of the entries padded to the longest rank; every rank
    then places the entries of rank r's particle i behind the global offset of i.
    Returns (offset [n + 1] int64, nbr [total] of nbr's dtype)."""
    import torch

    n = count.shape[0]
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        off = torch.zeros(n + 1, dtype=torch.int64, device=count.device)
        off[1:] = torch.cumsum(count, 0)
        return off, nbr
    world = dist.get_world_size()
    counts = [torch.empty_like(count) for _ in range(world)]
    dist.all_gather(counts, count.contiguous())
    total = torch.stack(counts).sum(0)
    off = torch.zeros(n + 1, dtype=torch.int64, device=count.device)
    off[1:] = torch.cumsum(total, 0)
    lens = torch.stack([c.sum() for c in counts])
    pad = int(lens.max().item())
    mine = torch.zeros(max(pad, 1), dtype=nbr.dtype, device=nbr.device)
    mine[: nbr.shape[0]] = nbr
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    out = torch.empty(int(off[-1].item()), dtype=nbr.dtype, device=nbr.device)
    for c, part in zip(counts, parts):
        t = int(c.sum().item())
        if t == 0:
            continue
        local_off = torch.cumsum(c, 0) - c
        dst = torch.repeat_interleave(off[:-1] - local_off, c) + torch.arange(t, dtype=torch.int64, device=c.device)
        out[dst] = part[:t]
    return off, out


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
