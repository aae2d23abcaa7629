"""Boundary behaviour of the C ABI on the GPU: error codes, call order, capacity, edge sizes, device I/O."""
import numpy as np
import pytest

from paper_1506_04553_b200 import workloads
from p3t_parity_helpers import assert_same_neighbour_sets, csr_sets, rel_err, widen

pytestmark = pytest.mark.gpu


def _binding():
    from paper_1506_04553_b200 import binding

    return binding


def test_call_order_and_argument_errors():
    b = _binding()
    cfg = workloads.config(1, n=512)
    with b.P3T(512, key_bits=30) as ctx:
        for call in (ctx.build_tree, ctx.eval_soft, ctx.get_acc_pot, ctx.get_neighbours):
            with pytest.raises(b.P3TError) as e:
                call()
            assert e.value.status == b.ESTATE
        ctx.load_particles(cfg["mass"], cfg["pos"])
        with pytest.raises(b.P3TError) as e:
            ctx.build_tree()                                    # parameters not set
        assert e.value.status == b.ESTATE
        for bad in [(-1.0, 0.5, 0.001, 0.01, 0.012), (1e-3, -0.1, 0.001, 0.01, 0.012), (1e-3, 0.5, 0.01, 0.01, 0.012),
                    (1e-3, 0.5, 0.001, 0.01, 0.009), (1e-3, 0.5, -0.001, 0.01, 0.012), (float("nan"), 0.5, 0.001, 0.01, 0.012)]:
            with pytest.raises(b.P3TError) as e:
                ctx.set_params(*bad)
            assert e.value.status == b.EINVAL
        with pytest.raises(b.P3TError):
            ctx.set_tree_params(0, 64)
        with pytest.raises(b.P3TError):
            ctx.set_tree_params(16, 48)
        ctx.set_params(cfg["eps"], 0.5, cfg["r_in"], cfg["r_out"], cfg["r_search"])
        ctx.build_tree()
        ctx.eval_soft()
        ctx.get_acc_pot()
        ctx.set_params(cfg["eps"], 0.6, cfg["r_in"], cfg["r_out"], cfg["r_search"])   # invalidates the tree
        with pytest.raises(b.P3TError) as e:
            ctx.eval_soft()
        assert e.value.status == b.ESTATE
        big = workloads.config(1, n=513)
        with pytest.raises(b.P3TError) as e:
            ctx.load_particles(big["mass"], big["pos"])         # n > max_n
        assert e.value.status == b.EINVAL
        bad = cfg["pos"].copy(); bad[7, 1] = np.inf
        with pytest.raises(b.P3TError) as e:
            ctx.load_particles(cfg["mass"], bad)
        assert e.value.status == b.EINVAL
    with pytest.raises(b.P3TError):
        b.P3T(512, key_bits=31)


def test_nonfinite_device_input_is_reported():
    import torch

    b = _binding()
    cfg = workloads.config(1, n=512)
    pos = torch.from_numpy(cfg["pos"]).cuda()
    pos[3, 2] = float("nan")
    with b.P3T(512, key_bits=63) as ctx:
        ctx.set_params(cfg["eps"], 0.5, cfg["r_in"], cfg["r_out"], cfg["r_search"])
        ctx.load_particles(torch.from_numpy(cfg["mass"]).cuda(), pos)
        with pytest.raises(b.P3TError) as e:
            ctx.synchronize()
        assert e.value.status == b.EINVAL


def test_neighbour_capacity_error_reports_total(oracle):
    b = _binding()
    cfg = workloads.config(1, n=2048)
    r_in, r_out, h = 0.01, 0.1, 0.12
    m, q = widen(cfg)
    ooff, olst, band = oracle.neighbours(q, cfg["eps"], h)
    want = int(ooff[-1])
    assert want > 1000 and len(band) == 0
    with b.P3T(2048, key_bits=63, nbr_capacity=100) as ctx:
        ctx.set_params(cfg["eps"], 0.5, r_in, r_out, h)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        with pytest.raises(b.P3TError) as e:
            ctx.get_neighbours()
        assert e.value.status == b.ECAPACITY
        count, total = ctx.get_neighbour_counts()
        assert total == want and np.array_equal(count.astype(np.int64), np.diff(ooff))
        acc, pot = ctx.get_acc_pot()                            # forces are unaffected
        a, p = oracle.direct(m, q, cfg["eps"], r_in, r_out)
        assert np.median(rel_err(acc.astype(np.float64), a)) < 1e-3
    with b.P3T(2048, key_bits=63, nbr_capacity=want) as ctx:    # retry with the reported total
        ctx.set_params(cfg["eps"], 0.5, r_in, r_out, h)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        off, nbr = ctx.get_neighbours()
        assert_same_neighbour_sets(csr_sets(off, nbr), csr_sets(ooff, olst), band)
        with pytest.raises(b.P3TError) as e:
            ctx.get_neighbours(capacity=want - 1)               # caller's buffer too small
        assert e.value.status == b.ECAPACITY


@pytest.mark.parametrize("n", [1, 2, 3, 31, 32, 33, 63, 64, 65, 257, 2049])
@pytest.mark.parametrize("theta", [0.0, 0.7])
def test_small_and_ragged_sizes(oracle, n, theta):
    b = _binding()
    cfg = workloads.config(1, n=max(n, 8))
    mass, pos = cfg["mass"][:n].copy(), np.ascontiguousarray(cfg["pos"][:n])
    r_in, r_out, h = 0.02, 0.2, 0.25
    with b.P3T(max(n, 1), key_bits=63) as ctx:
        ctx.set_params(1e-3, theta, r_in, r_out, h)
        ctx.soft_force(mass, pos)
        acc, pot = ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
    if n == 1:
        assert not acc.any() and pot[0] == 0.0 and off.tolist() == [0, 0]
        return
    a, p = oracle.direct(mass.astype(np.float64), pos.astype(np.float64), np.float32(1e-3), np.float32(r_in), np.float32(r_out))
    scale = np.abs(a).max()
    tol = 1e-5 if theta == 0.0 else 2e-2
    assert np.max(np.linalg.norm(acc - a, axis=1)) <= tol * scale
    ooff, olst, band = oracle.neighbours(pos.astype(np.float64), np.float32(1e-3), np.float32(h))
    assert_same_neighbour_sets(csr_sets(off, nbr), csr_sets(ooff, olst), band)


def test_device_pointers_in_and_out(oracle):
    import torch

    b = _binding()
    cfg = workloads.config(1, n=3000)
    with b.P3T(3000, key_bits=63) as ctx:
        ctx.set_walk_mode(1)      # bitwise comparison of two evaluations: one warp per group
        ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
        ctx.soft_force(cfg["mass"], cfg["pos"])
        acc_h, pot_h = ctx.get_acc_pot()
        ctx.soft_force(torch.from_numpy(cfg["mass"]).cuda(), torch.from_numpy(cfg["pos"]).cuda())
        acc_d, pot_d = ctx.get_acc_pot(on_device=True)
        torch.cuda.synchronize()
        assert np.array_equal(acc_d.cpu().numpy(), acc_h) and np.array_equal(pot_d.cpu().numpy(), pot_h)


def test_results_are_deterministic_and_context_reusable():
    b = _binding()
    c1, c2 = workloads.config(1, n=4096), workloads.config(3, n=3000)
    with b.P3T(4096, key_bits=63) as ctx:
        ctx.set_walk_mode(1)      # one warp per group: bitwise reproducible (include/p3t.h)
        outs = []
        for cfg in (c1, c2, c1):
            ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], 10 * cfg["r_out"], 12 * cfg["r_out"])
            ctx.soft_force(cfg["mass"], cfg["pos"])
            outs.append((ctx.get_acc_pot(), ctx.get_neighbours()))
        (a0, p0), (o0, n0) = outs[0]
        (a2, p2), (o2, n2) = outs[2]
        assert np.array_equal(a0, a2) and np.array_equal(p0, p2) and np.array_equal(o0, o2) and np.array_equal(n0, n2)


@pytest.mark.parametrize("n", [777, 20011, 150000])
def test_cooperative_and_split_walks_match_one_warp_per_group(n):
    """p3t_set_walk_mode: the CTA-per-group walk and the split walks (2 or 4 warps per group, each taking every 2nd /
    4th cell of one tree level) evaluate the same interactions (counts, neighbour lists identical); sums differ only by
    the fp32 rounding of differently composed batches."""
    b = _binding()
    cfg = workloads.config(1, n=n)
    with b.P3T(n, key_bits=63, nbr_capacity=256 * n) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], 10 * cfg["r_out"], 12 * cfg["r_out"])
        out = {}
        for mode in (1, 2, 3, 4, 0):
            ctx.set_walk_mode(mode)
            ctx.soft_force(cfg["mass"], cfg["pos"])
            st = ctx.get_stats()
            out[mode] = (ctx.get_acc_pot(), ctx.get_neighbours(), (st["n_pp"], st["n_pc"], st["n_near"], st["n_neighbours"]))
            if mode in (3, 4):      # the split walk adds its parts in a fixed order: bitwise reproducible
                ctx.soft_force(cfg["mass"], cfg["pos"])
                a_again, p_again = ctx.get_acc_pot()
                assert np.array_equal(a_again, out[mode][0][0]) and np.array_equal(p_again, out[mode][0][1])
        (a1, p1), (o1, l1), c1 = out[1]
        for mode in (2, 3, 4, 0):
            (a2, p2), (o2, l2), c2 = out[mode]
            assert c1 == c2 and np.array_equal(o1, o2) and np.array_equal(l1, l2)
            rel = np.linalg.norm(a1 - a2, axis=1) / np.linalg.norm(a1, axis=1)
            assert rel.max() <= 5e-6 and np.abs(p2 / p1 - 1).max() <= 2e-6
        with pytest.raises(b.P3TError):
            ctx.set_walk_mode(5)


def test_group_order_is_a_permutation_by_decreasing_cost_and_changes_nothing():
    """The schedule of a walk (its groups by decreasing predicted cost: the cost class the group of each group's first
    body had in the previous call) is a permutation of the groups; with unchanged positions it is sorted by the cost the
    header defines up to the cost classes (eight per octave); and it leaves the results bitwise alike."""
    b = _binding()
    cfg = workloads.config(3, n=60000)
    with b.P3T(cfg["n"], key_bits=63) as ctx:
        ctx.set_walk_mode(1)
        ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
        ctx.soft_force(cfg["mass"], cfg["pos"])          # no history: one class, any order
        a0, p0 = ctx.get_acc_pot()
        gs = ctx.array("group_start").astype(np.int64)
        ng = len(gs) - 1
        assert np.array_equal(np.sort(ctx.array("group_order").astype(np.int64)), np.arange(ng))
        ctx.soft_force(cfg["mass"], cfg["pos"])          # same tree: groups handed out by the costs of the first call
        a1, p1 = ctx.get_acc_pot()
        assert np.array_equal(a0, a1) and np.array_equal(p0, p1)
        order = ctx.array("group_order").astype(np.int64)
        stats = ctx.array("group_stats").astype(np.int64)
        assert np.array_equal(np.sort(order), np.arange(ng))
        cost = (13 * stats[:, 0] + 33 * stats[:, 1]) * np.where(np.diff(gs) > 32, 2, 1)
        bits = np.maximum(cost, 1).astype(np.float32).view(np.uint32).astype(np.int64) >> 20    # 8 classes per octave
        assert np.all(np.diff(bits[order]) <= 0) and bits[order][0] > bits[order][-1]
        # moved positions: another tree, other group numbers -- still a permutation, still close to cost order
        rng = np.random.default_rng(3)
        pos2 = (cfg["pos"] + 1e-3 * rng.normal(size=cfg["pos"].shape)).astype(np.float32)
        ctx.soft_force(cfg["mass"], pos2)
        order = ctx.array("group_order").astype(np.int64)
        stats = ctx.array("group_stats").astype(np.int64)
        gs = ctx.array("group_start").astype(np.int64)
        ng = len(gs) - 1
        assert np.array_equal(np.sort(order), np.arange(ng))
        cost = (13 * stats[:, 0] + 33 * stats[:, 1]) * np.where(np.diff(gs) > 32, 2, 1)
        rank = np.empty(ng); rank[order] = np.arange(ng)
        from scipy.stats import spearmanr
        assert spearmanr(rank, -cost).correlation > 0.8       # predicted order follows the measured cost


def test_all_bodies_at_one_point_and_massless_bodies(oracle):
    b = _binding()
    n = 100
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    pos = np.zeros((n, 3), dtype=np.float32) + np.float32(0.25)
    with b.P3T(n, key_bits=63) as ctx:
        ctx.set_params(1e-2, 0.5, 0.001, 0.005, 0.005)          # r_out < eps: plain softened Newton
        ctx.soft_force(mass, pos)
        acc, pot = ctx.get_acc_pot()
        assert not acc.any()
        np.testing.assert_allclose(pot, -(n - 1) / n / np.float32(1e-2), rtol=1e-6)
        assert ctx.get_neighbour_counts()[1] == 0
    cfg = workloads.config(1, n=1000)
    mass = cfg["mass"].copy(); mass[::3] = 0.0
    with b.P3T(1000, key_bits=30) as ctx:
        ctx.set_params(cfg["eps"], 0.5, cfg["r_in"], cfg["r_out"], cfg["r_search"])
        ctx.soft_force(mass, cfg["pos"])
        acc, pot = ctx.get_acc_pot()
        a, p = oracle.direct(mass.astype(np.float64), cfg["pos"].astype(np.float64), cfg["eps"], cfg["r_in"], cfg["r_out"])
        assert np.median(rel_err(acc.astype(np.float64), a)) < 1e-3


@pytest.mark.parametrize("world,mode", [(2, 1), (3, 1), (4, 2)])
def test_sharded_evaluations_add_up_to_the_whole(world, mode):
    """p3t_set_shard: the ranks' results (run one after the other on this GPU) combine to the unsharded evaluation:
    every particle is produced by exactly one rank, bitwise the same with one warp per group."""
    from paper_1506_04553_b200 import multi

    b = _binding()
    cfg = workloads.config(3, n=50000)
    n = cfg["n"]
    with b.P3T(n, key_bits=63, nbr_capacity=64 * n) as ctx:
        ctx.set_walk_mode(mode)
        ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], 10 * cfg["r_out"], 12 * cfg["r_out"])
        ctx.soft_force(cfg["mass"], cfg["pos"])
        a_full, p_full = ctx.get_acc_pot()
        o_full, l_full = ctx.get_neighbours()
        full = ctx.get_stats()
        accs, pots, csrs, npp = [], [], [], 0
        for r in range(world):
            ctx.set_shard(r, world)
            ctx.soft_force(cfg["mass"], cfg["pos"])
            a, p = ctx.get_acc_pot()
            accs.append(a); pots.append(p); csrs.append(ctx.get_neighbours())
            st = ctx.get_stats()
            npp += st["n_pp"] + st["n_pc"]
        owners = sum((np.abs(p) > 0).astype(np.int64) for p in pots)
        assert np.all(owners == 1)                                   # phi < 0 for every particle of a cluster
        assert npp == full["n_pp"] + full["n_pc"]
        a, p = multi.merge_forces(accs), multi.merge_forces(pots)
        off, nbr = multi.merge_csr(csrs, n)
        assert np.array_equal(off, o_full) and np.array_equal(nbr, l_full)
        if mode == 1:
            assert np.array_equal(a, a_full) and np.array_equal(p, p_full)
        else:
            assert np.abs(p / p_full - 1).max() <= 2e-6
        with pytest.raises(b.P3TError):
            ctx.set_shard(2, 2)


def test_sharded_walks_with_exchanged_cost_classes_deal_the_same_order_to_every_rank():
    """p3t_get_shard_record / p3t_put_shard_classes: after the ranks (here: three contexts on this GPU, one after the
    other) have summed their records, every context holds every particle's cost class, orders the groups alike
    (atomic-free order kernel) and takes every third position of that order: each group has exactly one owner, the union
    is bitwise the unsharded result, and each rank's groups are a fair share of the predicted cost."""
    import torch
    from paper_1506_04553_b200 import multi

    b = _binding()
    cfg = workloads.config(3, n=60000)
    n, world = cfg["n"], 3
    with b.P3T(n, key_bits=63, nbr_capacity=64 * n) as full:
        full.set_walk_mode(1)
        full.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], 10 * cfg["r_out"], 12 * cfg["r_out"])
        full.soft_force(cfg["mass"], cfg["pos"])
        a_full, p_full = full.get_acc_pot()
        o_full, l_full = full.get_neighbours()
        gstats = full.array("group_stats")
    ctxs = []
    for r in range(world):
        c = b.P3T(n, key_bits=63, nbr_capacity=64 * n)
        c.set_walk_mode(1)
        c.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], 10 * cfg["r_out"], 12 * cfg["r_out"])
        c.set_shard(r, world)
        ctxs.append(c)
    for call in range(3):
        recs = []
        for c in ctxs:
            c.soft_force(cfg["mass"], cfg["pos"])
            recs.append(c.get_shard_record())
        total = torch.stack(recs).sum(0)
        owners = torch.stack([(r[:, 4] > 0).to(torch.int32) for r in recs]).sum(0)
        assert bool((owners == 1).all())                                   # every particle produced by exactly one rank
        acc, pot = total[:, :3].cpu().numpy(), total[:, 3].cpu().numpy()
        assert np.array_equal(acc, a_full) and np.array_equal(pot, p_full)
        off, nbr = multi.merge_csr([c.get_neighbours() for c in ctxs], n)
        assert np.array_equal(off, o_full) and np.array_equal(nbr, l_full)
        if call > 0:      # the walks of this call used the order made from the exchanged classes
            orders = [c.array("group_order") for c in ctxs]
            assert all(np.array_equal(orders[0], o) for o in orders[1:])
            cost = 13.0 * gstats[:, 0] + 33.0 * gstats[:, 1]
            by_rank = [cost[orders[0][r::world]].sum() for r in range(world)]
            assert max(by_rank) <= 1.02 * min(by_rank), by_rank              # positions of a cost-sorted order, dealt round robin
            assert cost[orders[0][:50]].mean() > 3 * cost[orders[0][-50:]].mean()   # longest first
        for c in ctxs:
            c.put_shard_classes(total)
    for c in ctxs:
        c.close()


def test_host_fetch_of_forces_is_the_same_after_other_calls_on_the_stream():
    """p3t_get_acc_pot to host buffers runs on the context's side stream behind the walk-end event of the last
    evaluation; calls that queue more work on the context's stream in between (the hard force from host velocities,
    which stages them in the arrays the unpack uses; a whole step from device state, whose last kick reads the forces)
    must not change what it returns, in whatever order the fetches come."""
    import torch

    from paper_1506_04553_b200 import binding

    cfg = workloads.config(1, n=20000)
    n = cfg["n"]
    vel = np.ascontiguousarray(cfg["vel"].astype(np.float32))
    with binding.P3T(n, key_bits=63, nbr_capacity=1 << 20) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], 0.1 * 0.02, 0.02, 0.025)
        ctx.set_walk_mode(1)       # one warp per group: bitwise reproducible (the cooperative walk this size would get by
                                   # default shares its stack between warps as they come, so its rounding varies from run to run)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        acc0, pot0 = ctx.get_acc_pot()                       # straight after the evaluation
        a1, p1 = ctx.get_acc_pot(on_device=True)             # the device form (context's stream)
        assert np.array_equal(a1.cpu().numpy(), acc0) and np.array_equal(p1.cpu().numpy(), pot0)
        off0, nbr0 = ctx.get_neighbours()
        ctx.eval_hard(vel)                                   # host velocities: staged where the unpack writes
        acc2, pot2 = ctx.get_acc_pot()
        assert np.array_equal(acc2, acc0) and np.array_equal(pot2, pot0)
        off2, nbr2 = ctx.get_neighbours()
        assert np.array_equal(off2, off0) and np.array_equal(nbr2, nbr0)
        # a whole step from device state, then the fetch of the NEW forces to the host without a synchronisation in between
        m = torch.from_numpy(cfg["mass"]).cuda()
        q = torch.from_numpy(cfg["pos"].astype(np.float64)).cuda()
        v = torch.from_numpy(cfg["vel"].astype(np.float64)).cuda()
        ctx.step(m, q, v, 1.0 / 1024, a0=0.1 * float(cfg["mass"][0]) / 0.02 ** 2)
        acc3, pot3 = ctx.get_acc_pot()
        a3, p3 = ctx.get_acc_pot(on_device=True)
        torch.cuda.synchronize()
        assert np.array_equal(a3.cpu().numpy(), acc3) and np.array_equal(p3.cpu().numpy(), pot3)
        # and they are the forces at the new positions: a fresh context agrees bitwise
        qn = q.cpu().numpy().astype(np.float32)
    with binding.P3T(n, key_bits=63, nbr_capacity=1 << 20) as ctx2:
        ctx2.set_params(cfg["eps"], cfg["theta"], 0.1 * 0.02, 0.02, 0.025)
        ctx2.set_walk_mode(1)
        ctx2.soft_force(cfg["mass"], np.ascontiguousarray(qn))
        acc4, pot4 = ctx2.get_acc_pot()
    assert np.array_equal(acc4, acc3) and np.array_equal(pot4, pot3)
