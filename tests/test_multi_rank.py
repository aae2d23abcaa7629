"""N > 1 launch logic on CPU: two processes over gloo (rendezvous on 127.0.0.1).

The soft-force path does not shard (one cluster per GPU, no data-path collective);
what ranks exchange is only the timing reduction of bench.py, which lives in paper_1506_04553_b200/multi.py.
"""
import os
import socket

import numpy as np
import pytest

from paper_1506_04553_b200 import multi, workloads


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = multi.rank_config(1, rank, n=512)
        fake_ms = [3.0, 5.0][rank]           # rank 1 is the slow one
        units, ms = multi.aggregate(dist, cfg["n"], fake_ms)
        dist.barrier()
        q.put((rank, units, ms, float(cfg["pos"][0, 0]), cfg["n"], cfg["theta"]))
    finally:
        dist.destroy_process_group()


def test_two_ranks_over_gloo_aggregate_units_and_take_the_slowest_time():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, u0, ms0, x0, n0, th0), (r1, u1, ms1, x1, n1, th1) = out
    assert (u0, u1) == (1024, 1024) and ms0 == ms1 == 5.0          # sum of units, max of times, same on every rank
    assert n0 == n1 == 512 and th0 == th1                          # weak scaling: same problem size and parameters
    assert x0 != x1                                                # but an independent cluster per rank
    assert multi.throughput(u0, ms0) == pytest.approx(1024 / 5e-3)


def test_rank_zero_is_the_single_gpu_workload_and_single_process_needs_no_backend():
    a, b = multi.rank_config(1, 0, n=256), workloads.config(1, n=256)
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["mass"], b["mass"])
    assert multi.aggregate(None, 256, 2.5) == (256, 2.5)
    c = multi.rank_config(4, 1, n=256)                             # King model keeps its own generator
    assert c["pos"].shape == (256, 3) and not np.array_equal(c["pos"], multi.rank_config(4, 0, n=256)["pos"])


def _shard_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = 10
        owner = np.arange(n) % world                      # particle i is produced by rank i % world
        acc = np.where((owner == rank)[:, None], np.arange(3 * n, dtype=np.float32).reshape(n, 3) + 1, 0).astype(np.float32)
        pot = np.where(owner == rank, -np.arange(n, dtype=np.float32) - 1, 0).astype(np.float32)
        cnt = np.where(owner == rank, np.arange(n) % 3, 0)
        off = np.zeros(n + 1, dtype=np.uint64); off[1:] = np.cumsum(cnt)
        nbr = np.concatenate([np.full(c, 100 * i, dtype=np.uint32) + np.arange(c, dtype=np.uint32) for i, c in enumerate(cnt)] + [np.zeros(0, np.uint32)])
        ta, tp = torch.from_numpy(acc.copy()), torch.from_numpy(pot.copy())
        multi.allreduce_forces(dist, ta, tp)
        goff, gnbr = multi.allgather_csr(dist, off, nbr, n)
        q.put((rank, ta.numpy(), tp.numpy(), goff, gnbr))
    finally:
        dist.destroy_process_group()


def test_sharded_results_combine_over_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=120) for _ in range(2)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    n = 10
    exp_acc = np.arange(3 * n, dtype=np.float32).reshape(n, 3) + 1
    exp_pot = -np.arange(n, dtype=np.float32) - 1
    cnt = np.arange(n) % 3
    exp_off = np.zeros(n + 1, dtype=np.uint64); exp_off[1:] = np.cumsum(cnt)
    exp_nbr = np.concatenate([np.full(c, 100 * i, dtype=np.uint32) + np.arange(c, dtype=np.uint32) for i, c in enumerate(cnt)])
    for rank, acc, pot, off, nbr in out:                  # every rank ends with the full result
        assert np.array_equal(acc, exp_acc) and np.array_equal(pot, exp_pot)
        assert np.array_equal(off, exp_off) and np.array_equal(nbr, exp_nbr)


def test_merge_csr_handles_empty_ranks():
    n = 4
    a = (np.array([0, 2, 2, 2, 3], dtype=np.uint64), np.array([7, 8, 9], dtype=np.uint32))
    b = (np.zeros(n + 1, dtype=np.uint64), np.zeros(0, dtype=np.uint32))
    c = (np.array([0, 0, 1, 1, 1], dtype=np.uint64), np.array([5], dtype=np.uint32))
    off, nbr = multi.merge_csr([a, b, c], n)
    assert off.tolist() == [0, 2, 3, 3, 4] and nbr.tolist() == [7, 8, 5, 9]


class _FakeShardCtx:
    """What multi.allreduce_shard needs of a context, on the CPU: the record of the particles this rank 'produced'."""

    def __init__(self, rank, world, n):
        import torch

        owner = np.arange(n) % world
        rec = np.zeros((n, 5), dtype=np.float32)
        mine = owner == rank
        rec[mine, :3] = np.arange(3 * n, dtype=np.float32).reshape(n, 3)[mine] + 1
        rec[mine, 3] = -np.arange(n, dtype=np.float32)[mine] - 1
        rec[mine, 4] = (np.arange(n)[mine] % 7) + 1          # cost class + 1
        self.rec = torch.from_numpy(rec)
        self.put = None

    def get_shard_record(self, rec=None):
        return self.rec.clone()

    def put_shard_classes(self, rec):
        self.put = rec.clone()


def _shard_tensor_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = 11
        ctx = _FakeShardCtx(rank, world, n)
        acc, pot = multi.allreduce_shard(dist, ctx)
        owner = np.arange(n) % world
        cnt = np.where(owner == rank, np.arange(n) % 4, 0).astype(np.int64)
        nbr = np.concatenate([np.full(c, 100 * i, dtype=np.int64) + np.arange(c) for i, c in enumerate(cnt)] + [np.zeros(0, np.int64)])
        off, lst = multi.allgather_csr_tensors(dist, torch.from_numpy(cnt), torch.from_numpy(nbr))
        q.put((rank, acc.numpy().copy(), pot.numpy().copy(), ctx.put.numpy().copy(), off.numpy(), lst.numpy()))
    finally:
        dist.destroy_process_group()


def test_one_allreduce_carries_forces_and_cost_classes_and_lists_travel_as_tensors():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_tensor_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=120) for _ in range(2)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    n = 11
    exp_acc = np.arange(3 * n, dtype=np.float32).reshape(n, 3) + 1
    exp_pot = -np.arange(n, dtype=np.float32) - 1
    cnt = np.arange(n) % 4
    exp_off = np.zeros(n + 1, dtype=np.int64); exp_off[1:] = np.cumsum(cnt)
    exp_nbr = np.concatenate([np.full(c, 100 * i, dtype=np.int64) + np.arange(c) for i, c in enumerate(cnt)])
    for rank, acc, pot, put, off, lst in out:
        assert np.array_equal(acc, exp_acc) and np.array_equal(pot, exp_pot)
        assert np.array_equal(put[:, 4], (np.arange(n) % 7) + 1)           # every rank got every particle's class back
        assert np.array_equal(off, exp_off) and np.array_equal(lst, exp_nbr)


def test_single_process_shard_helpers_need_no_backend():
    import torch

    ctx = _FakeShardCtx(0, 1, 5)
    acc, pot = multi.allreduce_shard(None, ctx)
    assert acc.shape == (5, 3) and pot.shape == (5,) and ctx.put is not None
    off, lst = multi.allgather_csr_tensors(None, torch.tensor([1, 0, 2]), torch.tensor([9, 4, 5]))
    assert off.tolist() == [0, 1, 1, 3] and lst.tolist() == [9, 4, 5]
