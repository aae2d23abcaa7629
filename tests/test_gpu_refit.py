"""GPU parity of the tree reuse row (first half; include/p3t.h p3t_refit_tree).

A refit keeps the sorted order, cells and groups of the last full build and makes bodies, moments, boxes and acceptance
radii again from the moved positions.  What must hold: the same tolerances against the direct sum as a fresh tree, the
same neighbour sets (exact), the old topology untouched, moments equal to the fp64 recomputation over the OLD body
ranges, and an acceptance radius that still bounds both clauses of R-MAC for bodies that left their cell's cube.
"""
import numpy as np
import pytest

from paper_1506_04553_b200 import workloads
from p3t_parity_helpers import assert_same_neighbour_sets, csr_sets, rel_err

pytestmark = pytest.mark.gpu

TOL_MEDIAN, TOL_P99 = 1e-3, 1e-2
TOPOLOGY = ["keys", "sorted_idx", "cell_meta", "cell_level", "cell_start", "cell_parent", "group_start", "root_cube"]


def _ctx(cfg, key_bits=None, **kw):
    from paper_1506_04553_b200 import binding

    ctx = binding.P3T(cfg["n"], key_bits=key_bits or cfg["key_bits"], **kw)
    ctx.set_tree_params(cfg["nleaf"], cfg["ngroup"])
    ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
    return ctx


def _check_lists(oracle, pos, eps, h, off, nbr):
    ooff, olst, band = oracle.neighbours(pos.astype(np.float64), eps, h)
    assert_same_neighbour_sets(csr_sets(off, nbr), csr_sets(ooff, olst), band)


@pytest.mark.parametrize("n,key_bits", [(16384, 30), (65536, 63)])
def test_config2_ten_calls_with_refits_on_calls_2_to_10(oracle, n, key_bits):
    cfg = workloads.config(2, n=n)
    m = cfg["mass"].astype(np.float64)
    pos, vel = cfg["pos"].copy(), cfg["vel"].copy()
    dt = np.float32(cfg["dt_soft"])
    with _ctx(cfg, key_bits=key_bits) as ctx:
        ctx.set_tree_reuse(16, 0.5, 1.0)               # never forced to rebuild: calls 2..10 are refits
        for step in range(10):
            ctx.load_particles(cfg["mass"], pos)
            ctx.refit_tree()
            st = ctx.get_stats()
            assert st["tree_refits"] == step           # call 1 is the build, every later one a refit of it
            ctx.eval_soft()
            acc, pot = ctx.get_acc_pot()
            if step in (0, 4, 9):
                a, p = oracle.direct(m, pos.astype(np.float64), cfg["eps"], cfg["r_in"], cfg["r_out"])
                e = rel_err(acc.astype(np.float64), a)
                assert np.median(e) <= TOL_MEDIAN and np.percentile(e, 99) <= TOL_P99, (step, np.median(e), np.percentile(e, 99))
                ep = np.abs(pot / p - 1)
                assert np.median(ep) <= TOL_MEDIAN and np.percentile(ep, 99) <= TOL_P99
                off, nbr = ctx.get_neighbours()
                _check_lists(oracle, pos, cfg["eps"], cfg["r_search"], off, nbr)
            vel = vel + dt * acc
            pos = np.ascontiguousarray(pos + dt * vel, dtype=np.float32)
        assert ctx.get_stats()["n_stray"] > 0          # after nine steps of 1/256 some bodies have left their leaves


def test_refit_keeps_the_topology_and_recomputes_moments_boxes_and_radii():
    from oracle import keytree

    cfg = workloads.config(3, n=30011)
    with _ctx(cfg) as ctx:
        ctx.set_tree_reuse(4, 0.25, 1.0)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        before = {k: ctx.array(k).copy() for k in TOPOLOGY}
        # a large move (a tenth of a crossing time): many bodies leave their cells
        pos = np.ascontiguousarray(cfg["pos"] + np.float32(0.05) * cfg["vel"], dtype=np.float32)
        ctx.load_particles(cfg["mass"], pos)
        ctx.refit_tree()
        st = ctx.get_stats()
        assert st["tree_refits"] == 1 and st["n_stray"] > 100
        for k in TOPOLOGY:
            assert np.array_equal(ctx.array(k), before[k]), k
        idx, keys, cube = before["sorted_idx"], before["keys"], before["root_cube"]
        bodies = ctx.array("bodies")
        assert np.array_equal(bodies[:, :3], pos[idx]) and np.array_equal(bodies[:, 3], cfg["mass"][idx])
        cells = keytree.build_cells(keys, 16, 21)
        mac, m0, m1 = ctx.array("cell_mac"), ctx.array("cell_mom0"), ctx.array("cell_mom1")
        bmin, bmax = ctx.array("cell_bmin"), ctx.array("cell_bmax")
        theta, h = cfg["theta"], cfg["r_search"]
        rng = np.random.default_rng(2)
        grown = 0
        for i in np.unique(np.concatenate([np.arange(64), rng.integers(0, len(cells), 1200)])):
            c = cells[i]
            M, com, Q, lo, hi = keytree.moments(bodies, c["start"], c["count"])
            ext = max(float((hi - lo).max()), 1e-30)
            assert abs(m0[i, 0] - M) <= 2e-6 * M
            np.testing.assert_allclose(mac[i, :3], com, atol=3e-6 * ext + 2e-7 * np.abs(com).max())
            np.testing.assert_allclose(np.concatenate([m0[i, 1:], m1[i, :3]]), Q, atol=2e-5 * M * ext * ext + 1e-30)
            assert np.array_equal(bmin[i, :3], lo.astype(np.float32)) and np.array_equal(bmax[i, :3], hi.astype(np.float32))
            g, l = keytree.cell_geometry(c, keys[c["start"]], cube[:3], cube[3], 21, curve="hilbert")
            # side of the smallest cube about the geometric centre that holds the bodies (= l while they are inside)
            lm = max(l, 2.0 * float(np.maximum(g - lo, hi - g).max()))
            grown += lm > l * (1 + 1e-6)
            delta = np.linalg.norm(com - g)
            rmax = np.linalg.norm(bodies[c["start"]:c["start"] + c["count"], :3].astype(np.float64) - com, axis=1).max()
            rc = np.sqrt(float(mac[i, 3]))
            assert rc >= (lm / theta + delta) * (1 - 1e-5)
            assert rc >= h + rmax
        assert grown > 50
        # the forces of the refitted tree meet the tolerances of a fresh one
        ctx.eval_soft()
        acc, pot = ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
        from oracle import p3t_oracle as O
        a, p = O.direct(cfg["mass"].astype(np.float64), pos.astype(np.float64), cfg["eps"], cfg["r_in"], cfg["r_out"])
        e = rel_err(acc.astype(np.float64), a)
        assert np.median(e) <= TOL_MEDIAN and np.percentile(e, 99) <= TOL_P99
        _check_lists(O, pos, cfg["eps"], cfg["r_search"], off, nbr)


def test_refit_rebuilds_when_it_must():
    cfg = workloads.config(1, n=5000)
    with _ctx(cfg, key_bits=63) as ctx:
        ctx.load_particles(cfg["mass"], cfg["pos"])
        ctx.refit_tree()                                  # default max_refits = 0: a build
        assert ctx.get_stats()["tree_refits"] == 0
        ctx.set_tree_reuse(2, 0.5, 0.02)
        pos = cfg["pos"].copy()
        counts = []
        for _ in range(5):
            pos = np.ascontiguousarray(pos + np.float32(1e-4) * cfg["vel"], dtype=np.float32)
            ctx.load_particles(cfg["mass"], pos)
            ctx.refit_tree()
            counts.append(ctx.get_stats()["tree_refits"])
        assert counts == [1, 2, 0, 1, 2]                  # a rebuild after max_refits refits
        # too many strays: rebuild at once
        ctx.set_tree_reuse(100, 0.5, 0.02)
        ctx.load_particles(cfg["mass"], pos)
        ctx.refit_tree()
        assert ctx.get_stats()["tree_refits"] == 3
        ctx.load_particles(cfg["mass"], np.ascontiguousarray(pos[::-1]))
        ctx.refit_tree()
        assert ctx.get_stats()["tree_refits"] == 0
        keys = ctx.array("keys")
        assert np.all(keys[1:] >= keys[:-1])
        # another n: no tree to reuse
        ctx.load_particles(cfg["mass"][:4000], pos[:4000])
        ctx.refit_tree()
        assert ctx.get_stats()["tree_refits"] == 0 and ctx.get_stats()["n_cells"] > 0
        # changed tree parameters: no tree to reuse
        ctx.set_tree_params(8, 32)
        ctx.load_particles(cfg["mass"][:4000], pos[:4000])
        ctx.refit_tree()
        assert ctx.get_stats()["tree_refits"] == 0
        ctx.eval_soft()
        # parameters of the cutoff may change between refits (they enter the acceptance radius, which is made again)
        ctx.set_params(cfg["eps"], 0.3, 0.002, 0.02, 0.025)
        ctx.load_particles(cfg["mass"][:4000], pos[:4000])
        ctx.refit_tree()
        assert ctx.get_stats()["tree_refits"] == 1
        ctx.eval_soft()
        from oracle import p3t_oracle as O
        a, p = O.direct(cfg["mass"][:4000].astype(np.float64), pos[:4000].astype(np.float64), cfg["eps"], 0.002, 0.02)
        acc, pot = ctx.get_acc_pot()
        e = rel_err(acc.astype(np.float64), a)
        assert np.median(e) <= TOL_MEDIAN and np.percentile(e, 99) <= TOL_P99
        off, nbr = ctx.get_neighbours()
        _check_lists(O, pos[:4000], cfg["eps"], 0.025, off, nbr)


def test_whole_steps_with_tree_reuse_match_steps_with_rebuilds():
    """p3t_step with reuse switched on: positions and velocities equal to those of a run that
    rebuilds every step within the soft force's own tolerance (the two trees differ, the physics does not)."""
    import torch

    cfg = workloads.config(2, n=20000)
    T = cfg["dt_soft"]
    a0 = 0.1 * float(cfg["mass"].mean()) / cfg["r_out"] ** 2
    out = []
    for reuse in (0, 4):
        with _ctx(cfg) as ctx:
            ctx.set_tree_reuse(reuse, 0.5, 0.05)
            ctx.soft_force(cfg["mass"], cfg["pos"])
            q = torch.from_numpy(cfg["pos"].astype(np.float64)).cuda()
            v = torch.from_numpy(cfg["vel"].astype(np.float64)).cuda()
            md = torch.from_numpy(cfg["mass"]).cuda()
            refits = []
            for _ in range(6):
                ctx.step(md, q, v, T, a0=a0)
                refits.append(ctx.get_stats()["tree_refits"])
            off, nbr = ctx.get_neighbours()
            out.append((q.cpu().numpy(), v.cpu().numpy(), off.copy(), nbr.copy(), refits))
    assert out[0][4] == [0] * 6 and out[1][4] == [1, 2, 3, 4, 0, 1]
    # the lists are those of positions that agree to ~1e-8: identical unless a pair sits that close to h
    assert abs(len(out[0][3]) - len(out[1][3])) <= 4
    dq = np.abs(out[0][0] - out[1][0]).max()
    dv = np.abs(out[0][1] - out[1][1]).max()
    # six kicks of T with accelerations that agree to ~1e-3 relative (median), |a| ~ 1
    assert dq <= 6 * T * T * 0.05 and dv <= 6 * T * 0.05, (dq, dv)
