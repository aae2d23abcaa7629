"""GPU parity of the pair-class row (include/p3t.h p3t_set_pair_classes) against
oracle part O8.

Same tolerances as the single-class path: neighbour sets identical to brute force (with the pair's own h; black holes
always list each other) outside the 1e-6 band, theta = 0 within 1e-5 per particle, workload theta median <= 1e-3 and
p99 <= 1e-2 and no worse than the CPU tree with classes; the hard force over the lists within 1e-7.
"""
import numpy as np
import pytest

from paper_1506_04553_b200 import workloads
from p3t_parity_helpers import assert_same_neighbour_sets, csr_sets, rel_err

pytestmark = pytest.mark.gpu

TOL_THETA0, TOL_MEDIAN, TOL_P99 = 1e-5, 1e-3, 1e-2


def _tab(oracle, cfg):
    cp = cfg["class_params"]
    return oracle.pair_table(cfg["eps"], cfg["r_in"], cfg["r_out"], cfg["r_search"], cp["r_in_bf"], cp["r_out_bf"],
                             cp["r_search_bf"], eps_bb=cp["eps_bb"])


def _ctx(cfg, theta=None, ngroup=None, walk_mode=0, **kw):
    from paper_1506_04553_b200 import binding

    ctx = binding.P3T(cfg["n"], key_bits=63, **kw)
    ctx.set_tree_params(cfg["nleaf"], ngroup or cfg["ngroup"])
    ctx.set_walk_mode(walk_mode)
    ctx.set_params(cfg["eps"], cfg["theta"] if theta is None else theta, cfg["r_in"], cfg["r_out"], cfg["r_search"])
    cp = cfg["class_params"]
    ctx.set_pair_classes(cfg["classes"], cp["r_in_bf"], cp["r_out_bf"], cp["r_search_bf"], cp["eps_bb"])
    return ctx


def _check_lists(oracle, cfg, tab, off, nbr):
    ooff, olst, band = oracle.neighbours_classes(cfg["pos"].astype(np.float64), cfg["classes"], tab)
    assert_same_neighbour_sets(csr_sets(off, nbr), csr_sets(ooff, olst), band)
    return ooff


def _smbh(n, extra_holes=0):
    """the paper's workload (two holes at (+-0.5, 0, 0)); extra holes are dropped into the core among the stars"""
    cfg = workloads.config(6, n=n)
    if extra_holes:
        k = np.argsort(np.linalg.norm(cfg["pos"], axis=1))[:extra_holes]
        cfg["classes"] = cfg["classes"].copy()
        cfg["classes"][k] = 1
        cfg["mass"] = cfg["mass"].copy()
        cfg["mass"][k] = 0.005
    return cfg


@pytest.mark.parametrize("ngroup,walk_mode", [(64, 1), (32, 2)])
def test_theta0_with_classes_is_the_direct_sum_with_classes(oracle, ngroup, walk_mode):
    cfg = _smbh(4094, extra_holes=3)
    tab = _tab(oracle, cfg)
    m, q = cfg["mass"].astype(np.float64), cfg["pos"].astype(np.float64)
    a, p = oracle.direct_classes(m, q, cfg["classes"], tab)
    with _ctx(cfg, theta=0.0, ngroup=ngroup, walk_mode=walk_mode) as ctx:
        ctx.soft_force(cfg["mass"], cfg["pos"])
        acc, pot = ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
        st = ctx.get_stats()
        assert st["n_pc"] == 0 and st["n_pp"] == cfg["n"] * (cfg["n"] - 1)
        assert rel_err(acc.astype(np.float64), a).max() <= TOL_THETA0
        assert np.max(np.abs(pot / p - 1)) <= TOL_THETA0
        ooff = _check_lists(oracle, cfg, tab, off, nbr)
        holes = np.flatnonzero(cfg["classes"] == 1)
        for i in holes:                                    # every hole lists every other hole (unsplit, L287)
            assert set(holes) - {i} <= set(nbr[int(off[i]):int(off[i + 1])].tolist())
        # the brute-force GPU entry gives the same
        ctx.eval_direct()
        accd, potd = ctx.get_acc_pot()
        offd, nbrd = ctx.get_neighbours()
        assert rel_err(accd.astype(np.float64), a).max() <= TOL_THETA0
        assert np.array_equal(offd, off) and np.array_equal(nbrd, nbr)


@pytest.mark.parametrize("n,extra,ngroup,walk_mode", [(16384, 0, 32, 0), (16384, 0, 64, 1), (30000, 5, 64, 1), (30000, 5, 32, 2),
                                                      (30000, 5, 64, 3), (20000, 3, 32, 4)])
def test_smbh_workload_at_theta_04(oracle, n, extra, ngroup, walk_mode):
    """16K Plummer + two m = 0.01 bodies at (+-0.5, 0, 0), r_cut,FS-FS = 1/256, r_cut,BH-FS = 1/32."""
    cfg = _smbh(n, extra_holes=extra)
    tab = _tab(oracle, cfg)
    m, q = cfg["mass"].astype(np.float64), cfg["pos"].astype(np.float64)
    a, p = oracle.direct_classes(m, q, cfg["classes"], tab)
    tree = oracle.Tree(m, q, nleaf=16)
    o4 = tree.walk_classes(cfg["classes"], tab, cfg["theta"])
    e4 = rel_err(o4["acc"], a)
    with _ctx(cfg, ngroup=ngroup, walk_mode=walk_mode) as ctx:
        ctx.soft_force(cfg["mass"], cfg["pos"])
        acc, pot = ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
        e = rel_err(acc.astype(np.float64), a)
        assert np.median(e) <= TOL_MEDIAN and np.percentile(e, 99) <= TOL_P99
        assert np.median(e) <= np.median(e4) * 1.05 + 2e-7 and np.percentile(e, 99) <= np.percentile(e4, 99) * 1.05 + 2e-7
        holes = np.flatnonzero(cfg["classes"] == 1)
        assert e[holes].max() <= TOL_P99                   # the holes' own soft force (no BH-BH part in it)
        ep = np.abs(pot / p - 1)
        assert np.median(ep) <= TOL_MEDIAN and np.percentile(ep, 99) <= TOL_P99
        ooff = _check_lists(oracle, cfg, tab, off, nbr)
        assert np.diff(ooff)[holes].min() >= len(holes) - 1
        # momentum: sum m a = 0 across the classes (pairwise antisymmetry; fp32 sums, tree error)
        scale = (m[:, None] * np.abs(a)).sum()
        assert np.abs((m[:, None] * acc).sum(0)).max() <= 2e-3 * scale
        # the hard part over these lists = O8's hard part over all pairs (BH-BH: the whole Newtonian term, eps_bb)
        ah, jh, ph = ctx.eval_hard(cfg["vel"])
        oa, oj, op = oracle.hard_classes(m, q, cfg["vel"].astype(np.float64), cfg["classes"], tab)
        busy = np.abs(oa).sum(1) > 0
        assert set(holes) <= set(np.flatnonzero(busy))
        # (a pair at the very edge of its cutoff sphere has 1 - K ~ 1e-12, a difference of O(1) numbers: the comparison is
        #  relative to the particle's own hard force, floored at 1e-4 of the typical one)
        na = np.linalg.norm(oa[busy], axis=1)
        nj = np.linalg.norm(oj[busy], axis=1)
        assert (np.linalg.norm(ah[busy] - oa[busy], axis=1) / np.maximum(na, 1e-4 * np.median(na))).max() <= 1e-7
        assert (np.linalg.norm(jh[busy] - oj[busy], axis=1) / np.maximum(nj, 1e-4 * np.median(nj))).max() <= 1e-6
        assert (np.abs(ph[busy] - op[busy]) / np.maximum(np.abs(op[busy]), 1e-4 * np.median(np.abs(op[busy])))).max() <= 1e-7
        assert not ah[~busy].any()
        # soft + hard = plain Newton for the holes (unsoftened between them, eps otherwise)
        for i in holes:
            d = q[i] - np.delete(q, i, axis=0)
            eps = np.where(np.delete(cfg["classes"], i) == 1, cfg["class_params"]["eps_bb"], cfg["eps"])
            newton = -(np.delete(m, i)[:, None] * d / ((d * d).sum(1) + eps ** 2)[:, None] ** 1.5).sum(0)
            assert np.linalg.norm(acc[i] + ah[i] - newton) <= 5e-3 * np.linalg.norm(newton)


def test_classes_all_zero_equal_no_classes_bitwise():
    cfg = workloads.config(6, n=8000)
    from paper_1506_04553_b200 import binding

    out = []
    for use in (False, True):
        with binding.P3T(cfg["n"], key_bits=63) as ctx:
            ctx.set_walk_mode(1)
            ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
            if use:
                ctx.set_pair_classes(np.zeros(cfg["n"], np.uint8), 0.01, 0.1, 0.12, 0.0)
            ctx.soft_force(cfg["mass"], cfg["pos"])
            acc, pot = ctx.get_acc_pot()
            off, nbr = ctx.get_neighbours()
            out.append((acc, pot, off, nbr, ctx.get_stats()))
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][3], out[1][3])
    assert out[0][4]["n_pp"] == out[1][4]["n_pp"] and out[0][4]["n_pc"] == out[1][4]["n_pc"]


def test_class_arguments_and_state():
    from paper_1506_04553_b200 import binding

    cfg = workloads.config(6, n=1000)
    with binding.P3T(cfg["n"], key_bits=63) as ctx:
        ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])
        bad = cfg["classes"].copy(); bad[3] = 2
        for args in [(bad, 0.01, 0.1, 0.12, 0.0), (cfg["classes"], 0.1, 0.1, 0.12, 0.0), (cfg["classes"], 0.01, 0.1, 0.05, 0.0),
                     (cfg["classes"], 0.01, 0.1, 0.12, -1.0), (cfg["classes"], -0.01, 0.1, 0.12, 0.0)]:
            with pytest.raises(binding.P3TError) as ei:
                ctx.set_pair_classes(*args)
            assert ei.value.status == binding.EINVAL
        ctx.set_pair_classes(cfg["classes"][:500], 0.01, 0.1, 0.12, 0.0)
        ctx.load_particles(cfg["mass"], cfg["pos"])
        with pytest.raises(binding.P3TError) as ei:
            ctx.build_tree()
        assert ei.value.status == binding.ESTATE
        cp = cfg["class_params"]
        import torch
        ctx.set_pair_classes(torch.from_numpy(cfg["classes"]).cuda(), cp["r_in_bf"], cp["r_out_bf"], cp["r_search_bf"], cp["eps_bb"])
        ctx.soft_force(cfg["mass"], cfg["pos"])
        off, nbr = ctx.get_neighbours()
        n = cfg["n"]
        assert n - 2 in nbr[int(off[n - 1]):int(off[n])].tolist()
        ctx.set_pair_classes(None)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        off, nbr = ctx.get_neighbours()
        assert n - 2 not in nbr[int(off[n - 1]):int(off[n])].tolist()
        ctx.hermite_step(cfg["pos"].astype(np.float64), cfg["vel"].astype(np.float64), 1e-3)


@pytest.mark.parametrize("n,extra,cluster_max", [(16384, 0, None), (20000, 6, None), (6000, 40, 64)])
def test_hermite_part_with_classes_takes_the_oracles_steps(oracle, n, extra, cluster_max):
    """p3t_hermite_step with pair classes against oracle O7-with-classes over the same lists: the two holes of the paper's
    SMBH start (each other's neighbours at distance 1: a pure Hermite pair, unsoftened) and the field stars within
    r_search,BH-FS of a hole; extra holes in the core make clusters with several holes (cluster_max = 64 sends the larger
    ones to the thread-block-cluster tier)."""
    cfg = _smbh(n, extra_holes=extra)
    tab = _tab(oracle, cfg)
    m, q, v = cfg["mass"].astype(np.float64), cfg["pos"].astype(np.float64), cfg["vel"].astype(np.float64)
    cls = cfg["classes"]
    T = cfg["dt_soft"]
    ooff, olst, band = oracle.neighbours_classes(q, cls, tab)
    assert len(band) == 0
    a0 = (0.1 * float(m[0]) / cfg["r_out"] ** 2, 0.1 * 0.01 / cfg["class_params"]["r_out_bf"] ** 2)
    eta, eta_s = (0.1, 0.03), (0.01, 0.003)
    oq, ov, oinfo = oracle.hermite_classes(m, q, v, cls, tab, ooff, olst, T, eta=eta, eta_s=eta_s, a0=a0)
    with _ctx(cfg, nbr_capacity=max(int(ooff[-1]) + 1024, 1 << 16)) as ctx:
        ctx.soft_force(cfg["mass"], cfg["pos"])
        off, nbr = ctx.get_neighbours()
        assert np.array_equal(off.astype(np.int64), ooff) and np.array_equal(nbr.astype(np.int64), olst.astype(np.int64))
        ctx.set_hermite_class_params(eta[1], eta_s[1], a0[1])
        if cluster_max:
            ctx.set_hermite_cluster_max(cluster_max)
        gq, gv = q.copy(), v.copy()
        info = ctx.hermite_step(gq, gv, T, eta=eta[0], eta_s=eta_s[0], a0=a0[0])
    holes = np.flatnonzero(cls == 1)
    assert info["n_steps"] == int(oinfo["nstep"].sum()) and oinfo["nstep"][holes].min() >= 4
    assert info["n_nonisolated"] == int((np.diff(ooff) > 0).sum())
    iso = np.diff(ooff) == 0
    assert np.array_equal(gq[iso], oq[iso])
    assert np.abs(gq - oq).max() <= 1e-9 * np.abs(T * v).max() and np.abs(gv - ov).max() <= 1e-9 * np.abs(v).max()
    # the holes moved under each other's pull, not on straight lines
    assert np.abs(gq[holes] - (q[holes] + T * v[holes])).max() > 1e-12


def test_whole_steps_with_classes_conserve_energy():
    """p3t_step on the paper's SMBH start: 16 steps; the total energy (kinetic + the kinds' own softened potentials by a
    direct sum in numpy) stays within the soft force's tolerance."""
    import torch

    cfg = _smbh(8192)
    m, cls = cfg["mass"].astype(np.float64), cfg["classes"]
    T = cfg["dt_soft"]

    def energy(q, v):
        d = q[:, None, :] - q[None, :, :]
        eps = np.where((cls[:, None] == 1) & (cls[None, :] == 1), cfg["class_params"]["eps_bb"], cfg["eps"])
        s = np.sqrt((d * d).sum(-1) + eps ** 2)
        np.fill_diagonal(s, np.inf)
        return 0.5 * (m * (v * v).sum(1)).sum() - 0.5 * (m[:, None] * m[None, :] / s).sum()

    q0, v0 = cfg["pos"].astype(np.float64), cfg["vel"].astype(np.float64)
    e0 = energy(q0, v0)
    with _ctx(cfg) as ctx:
        ctx.set_hermite_class_params(0.03, 0.003, 0.1 * 0.01 / cfg["class_params"]["r_out_bf"] ** 2)
        ctx.soft_force(cfg["mass"], cfg["pos"])
        q, v = torch.from_numpy(q0).cuda(), torch.from_numpy(v0).cuda()
        md = torch.from_numpy(cfg["mass"]).cuda()
        for _ in range(16):
            info = ctx.step(md, q, v, T, a0=0.1 * float(m[0]) / cfg["r_out"] ** 2)
        assert info["n_nonisolated"] >= 2
    e1 = energy(q.cpu().numpy(), v.cpu().numpy())
    assert abs(e1 / e0 - 1) < 2e-4, (e0, e1)


def test_refit_with_classes_keeps_lists_exact(oracle):
    """Tree reuse with pair classes: the class bytes in key order and the black-hole flags of the cells are those of the
    last build; boxes and radii are remade from the moved positions, so the lists (kind by kind) stay exact."""
    cfg = _smbh(20000, extra_holes=4)
    tab = _tab(oracle, cfg)
    m = cfg["mass"].astype(np.float64)
    with _ctx(cfg, walk_mode=1) as ctx:
        ctx.set_tree_reuse(4, 0.5, 1.0)
        pos = cfg["pos"].copy()
        for call in range(3):
            ctx.load_particles(cfg["mass"], pos)
            ctx.refit_tree()
            assert ctx.get_stats()["tree_refits"] == call
            ctx.eval_soft()
            acc, pot = ctx.get_acc_pot()
            off, nbr = ctx.get_neighbours()
            q = pos.astype(np.float64)
            a, p = oracle.direct_classes(m, q, cfg["classes"], tab)
            e = rel_err(acc.astype(np.float64), a)
            assert np.median(e) <= TOL_MEDIAN and np.percentile(e, 99) <= TOL_P99
            ooff, olst, band = oracle.neighbours_classes(q, cfg["classes"], tab)
            assert_same_neighbour_sets(csr_sets(off, nbr), csr_sets(ooff, olst), band)
            pos = np.ascontiguousarray(pos + np.float32(4 * cfg["dt_soft"]) * cfg["vel"], dtype=np.float32)
