"""Pins for the oracle's Barnes-Hut tree (O4) and for the workload generators.

P12  theta = 0 equals the direct sum; tree neighbour lists equal O3 for every theta
P13  quadrupole error of a distant clump falls as (l/d)^3 (slope ~2 if Q is dropped)   L138
P14  moments: sum M_leaf = M, root COM, parent Q == Q recomputed from bodies; topology
P15  error decreases and interaction count grows as theta decreases                     L173-175, L193
The absolute error level at a given theta is NOT fixed by the paper (parity unpinned).
"""
import math

import numpy as np
import pytest

from paper_1506_04553_b200 import workloads


@pytest.fixture(scope="module")
def cfg():
    c = workloads.config(1, n=2048)
    c["m64"], c["q64"] = c["mass"].astype(np.float64), c["pos"].astype(np.float64)
    return c


def test_p12_theta0_is_direct_sum(oracle, cfg):
    r_in, r_out, h = 0.01, 0.1, 0.12     # stress radii: many pairs inside the cutoff
    a, p = oracle.direct(cfg["m64"], cfg["q64"], cfg["eps"], r_in, r_out)
    t = oracle.Tree(cfg["m64"], cfg["q64"], nleaf=8)
    r = t.walk(cfg["eps"], 0.0, r_in, r_out, h)
    np.testing.assert_allclose(r["acc"], a, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(r["pot"], p, rtol=1e-12)
    assert np.all(r["n_pp"] == cfg["n"] - 1) and np.all(r["n_pc"] == 0)


@pytest.mark.parametrize("theta", [0.0, 0.3, 0.8, 1.5])
def test_p12_tree_neighbours_equal_brute_force(oracle, cfg, theta):
    r_in, r_out, h = 0.01, 0.1, 0.12
    off, lst, _ = oracle.neighbours(cfg["q64"], cfg["eps"], h)
    t = oracle.Tree(cfg["m64"], cfg["q64"], nleaf=16)
    stride = int(np.diff(off).max())
    r = t.walk(cfg["eps"], theta, r_in, r_out, h, nbr_stride=stride)
    assert np.array_equal(r["nbr_count"], np.diff(off))
    for i in range(0, cfg["n"], 7):
        assert list(r["nbr"][i, : r["nbr_count"][i]]) == list(lst[off[i]:off[i + 1]])
    if theta > 0:
        # clause 3 of R-MAC: every pair closer than h was met in an opened leaf, so the tree
        # result's K/W-weighted part is exact; only far-field multipole error remains
        a, _ = oracle.direct(cfg["m64"], cfg["q64"], cfg["eps"], r_in, r_out)
        err = np.linalg.norm(r["acc"] - a, axis=1) / np.linalg.norm(a, axis=1)
        assert np.median(err) < 0.05


def test_p12_group_box_opens_superset(oracle, cfg):
    # the same targets walked with an enclosing box B open more and err less (R-MAC uses B)
    t = oracle.Tree(cfg["m64"], cfg["q64"])
    a, _ = oracle.direct(cfg["m64"], cfg["q64"], cfg["eps"], cfg["r_in"], cfg["r_out"])
    sub = np.arange(64)
    lo, hi = cfg["q64"][sub].min(0), cfg["q64"][sub].max(0)
    box = np.tile(np.concatenate([lo, hi]), (64, 1))
    r0 = t.walk(cfg["eps"], 0.6, cfg["r_in"], cfg["r_out"], cfg["r_search"], subset=sub)
    r1 = t.walk(cfg["eps"], 0.6, cfg["r_in"], cfg["r_out"], cfg["r_search"], subset=sub, box=box)
    assert np.all(r1["n_pp"] >= r0["n_pp"])
    e0 = np.linalg.norm(r0["acc"] - a[sub], axis=1) / np.linalg.norm(a[sub], axis=1)
    e1 = np.linalg.norm(r1["acc"] - a[sub], axis=1) / np.linalg.norm(a[sub], axis=1)
    assert np.median(e1) < np.median(e0)


def test_p13_quadrupole_error_slope(oracle):
    rng = np.random.default_rng(3)
    n = 64
    clump = rng.uniform(-0.5, 0.5, (n, 3))
    m = rng.uniform(0.5, 1.5, n + 1) / n
    m[-1] = 1e-30  # the probe
    u = np.array([0.48, -0.6, 0.64])

    def errors(use_quad):
        out = []
        for d in (8.0, 16.0, 32.0, 64.0):
            pos = np.vstack([clump, d * u])
            t = oracle.Tree(m, pos, nleaf=n, max_depth=1)   # root splits once: probe alone in its octant
            sub = np.array([n])
            # theta huge: every cell that does not contain the probe is accepted at once
            r = t.walk(0.0, 100.0, 1e-6, 1e-5, 2e-5, subset=sub, use_quad=use_quad)
            a, _ = oracle.direct(m, pos, 0.0, 1e-6, 1e-5, subset=sub)
            assert r["n_pp"][0] == 0
            out.append(np.linalg.norm(r["acc"] - a) / np.linalg.norm(a))
        return np.array(out)

    eq, em = errors(True), errors(False)
    slope_q = np.polyfit(np.log([8, 16, 32, 64]), np.log(eq), 1)[0]
    slope_m = np.polyfit(np.log([8, 16, 32, 64]), np.log(em), 1)[0]
    assert -3.4 < slope_q < -2.7      # octupole is the first neglected term
    assert -2.4 < slope_m < -1.7      # quadrupole is the first neglected term
    assert np.all(eq < em)


def _clump(seed=3, n=64):
    rng = np.random.default_rng(seed)
    clump = rng.uniform(-0.5, 0.5, (n, 3))
    m = rng.uniform(0.5, 1.5, n + 1) / n
    m[-1] = 1e-30  # the probe
    return n, clump, m


def test_p13_quadrupole_potential_error_slope(oracle):
    """R-QUAD's potential term (L138 "up to the quadrupole moment"): the relative error of phi against the
    exact sum falls as (l/d)^3 with Q and as (l/d)^2 without -- a wrong sign or factor in either half of
    -1/2 [3 RQR/s^5 - trQ/s^3] leaves a second-order error and fails the slope."""
    n, clump, m = _clump()
    # rms over five directions: along a single one the octupole can nearly vanish and spoil the fit
    us = np.array([[0.48, -0.6, 0.64], [0.6, 0.64, -0.48], [-0.64, 0.48, 0.6], [1.0, 0.0, 0.0], [0.0, 0.6, 0.8]])
    ds = (8.0, 16.0, 32.0, 64.0)

    def errors(use_quad, eps):
        out = []
        for d in ds:
            e2 = 0.0
            for u in us:
                pos = np.vstack([clump, d * u])
                t = oracle.Tree(m, pos, nleaf=n, max_depth=1)
                sub = np.array([n])
                r = t.walk(eps, 100.0, 1e-6, 1e-5, 2e-5, subset=sub, use_quad=use_quad)
                _, p = oracle.direct(m, pos, eps, 1e-6, 1e-5, subset=sub)
                assert r["n_pp"][0] == 0 and r["n_pc"][0] >= 1
                e2 += ((r["pot"][0] - p[0]) / p[0]) ** 2
            out.append(math.sqrt(e2 / len(us)))
        return np.array(out)

    for eps in (0.0, 0.7):      # softened cell terms carry the same eps (reading A8)
        eq, em = errors(True, eps), errors(False, eps)
        slope_q = np.polyfit(np.log(ds), np.log(eq), 1)[0]
        slope_m = np.polyfit(np.log(ds), np.log(em), 1)[0]
        assert -3.4 < slope_q < -2.7, (eps, slope_q)
        assert -2.4 < slope_m < -1.7, (eps, slope_m)
        assert np.all(eq < 0.2 * em)


def test_p13_cell_acceleration_is_minus_gradient_of_cell_potential(oracle):
    """a = -grad phi term by term for accepted cells: central differences of the walk's potential for a
    probe moved by +-delta, the accepted set frozen (theta huge, one split: every octant of the clump is
    accepted whole, the probe sits alone in its own), equal the walk's acceleration."""
    n, clump, m = _clump(seed=5)
    probe = np.array([2.9, -3.7, 4.3])
    for eps in (0.0, 0.9):
        def walk(p):
            pos = np.vstack([clump, p])
            t = oracle.Tree(m, pos, nleaf=n, max_depth=1)
            r = t.walk(eps, 100.0, 1e-6, 1e-5, 2e-5, subset=np.array([n]))
            assert r["n_pp"][0] == 0
            # signature of the decomposition: which bodies sit in which cell
            return r, (int(r["n_pc"][0]), t.nodes()["count"].tolist(), t.perm().tolist())
        r0, npc0 = walk(probe)
        delta = 1e-4
        grad = np.zeros(3)
        for ax in range(3):
            e = np.zeros(3); e[ax] = delta
            rp, npc_p = walk(probe + e)
            rm, npc_m = walk(probe - e)
            assert npc_p == npc_m == npc0          # same cells, same members: the accepted set is frozen
            grad[ax] = (rp["pot"][0] - rm["pot"][0]) / (2 * delta)
        np.testing.assert_allclose(r0["acc"][0], -grad, rtol=1e-6, atol=1e-6 * np.linalg.norm(grad))
        # and the quadrupole part is not negligible here: dropping Q moves the result far beyond that tolerance
        pos = np.vstack([clump, probe])
        t = oracle.Tree(m, pos, nleaf=n, max_depth=1)
        rq = t.walk(eps, 100.0, 1e-6, 1e-5, 2e-5, subset=np.array([n]), use_quad=False)
        assert abs(rq["pot"][0] - r0["pot"][0]) > 1e-4 * abs(r0["pot"][0])


def test_p14_moments_and_topology(oracle, cfg):
    m, q = cfg["m64"], cfg["q64"]
    t = oracle.Tree(m, q, nleaf=16)
    nd, perm = t.nodes(), t.perm()
    assert sorted(perm.tolist()) == list(range(cfg["n"]))
    assert nd["M"][nd["leaf"]].sum() == pytest.approx(m.sum(), rel=1e-13)
    assert nd["count"][nd["leaf"]].sum() == cfg["n"]
    np.testing.assert_allclose(nd["c"][0], (m[:, None] * q).sum(0) / m.sum(), atol=1e-13)
    for k in range(0, t.nnodes, 5):
        b = perm[nd["first"][k]: nd["first"][k] + nd["count"][k]]
        c = (m[b, None] * q[b]).sum(0) / m[b].sum()
        r = q[b] - c
        Q = np.array([(m[b] * r[:, i] * r[:, j]).sum() for i, j in ((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))])
        np.testing.assert_allclose(nd["c"][k], c, atol=1e-12)
        np.testing.assert_allclose(nd["Q"][k], Q, atol=1e-15, rtol=1e-9)
        np.testing.assert_allclose(nd["bmin"][k], q[b].min(0))
        np.testing.assert_allclose(nd["bmax"][k], q[b].max(0))
        half = 0.5 * nd["side"][k]
        assert np.all(np.abs(q[b] - nd["g"][k]) <= half * (1 + 1e-12))      # cube contains its bodies
        if not nd["leaf"][k]:
            ch = nd["child"][k][nd["child"][k] >= 0]
            assert nd["count"][ch].sum() == nd["count"][k] and nd["count"][k] > 16
            assert np.all(nd["level"][ch] == nd["level"][k] + 1)
        else:
            assert nd["count"][k] <= 16 or nd["level"][k] == 21


def test_p14_max_depth_leaf_may_exceed_nleaf(oracle):
    q = np.zeros((40, 3))
    q[20:] = 1.0
    m = np.full(40, 1 / 40)
    t = oracle.Tree(m, q, nleaf=4, max_depth=6)
    nd = t.nodes()
    assert nd["count"][nd["leaf"]].max() == 20 and nd["level"].max() == 6
    r = t.walk(0.1, 0.5, 0.01, 0.1, 0.12)    # coincident bodies interact (self excluded by index, A13)
    a, p = oracle.direct(m, q, 0.1, 0.01, 0.1)
    np.testing.assert_allclose(r["pot"], p, rtol=1e-3)
    assert np.all(r["nbr_count"] == 19)


def test_p15_error_and_cost_vs_theta(oracle, cfg):
    a, _ = oracle.direct(cfg["m64"], cfg["q64"], cfg["eps"], cfg["r_in"], cfg["r_out"])
    t = oracle.Tree(cfg["m64"], cfg["q64"])
    med, cost = [], []
    for theta in (0.8, 0.5, 0.4, 0.2):
        r = t.walk(cfg["eps"], theta, cfg["r_in"], cfg["r_out"], cfg["r_search"])
        e = np.linalg.norm(r["acc"] - a, axis=1) / np.linalg.norm(a, axis=1)
        med.append(np.median(e))
        cost.append((r["n_pp"] + r["n_pc"]).mean())
    assert all(x > y for x, y in zip(med, med[1:]))
    assert all(x < y for x, y in zip(cost, cost[1:]))
    assert med[2] < 1e-3   # theta = 0.4 (north_star's bar; reported, not fixed by the paper)


# ---------------------------------------------------------------- workloads (O5)
def test_workload_plummer_shape():
    pos, vel = workloads.plummer(20000, 7)
    r = np.linalg.norm(pos, axis=1)
    a = workloads.PLUMMER_A
    assert r.max() <= 20 * a
    # half-mass radius of a Plummer sphere: a / sqrt(2^(2/3) - 1) = 1.3048 a
    assert np.median(r) == pytest.approx(1.3048 * a, rel=0.03)
    # virial: T = 3 pi/(64 a) = 1/4 for M = 1
    assert 0.5 * (vel**2).sum(1).mean() == pytest.approx(0.25, rel=0.03)


def test_workload_salpeter():
    m = workloads.salpeter_masses(200000, 11)
    assert m.sum() == pytest.approx(1.0, rel=1e-12)
    assert m.max() / m.min() < 1000.0 + 1e-9
    # fraction of stars above 1 (in units of m_lo = 0.1 -> 10 m_lo): (10^-1.35 - 1000^-1.35)/(1 - 1000^-1.35)
    frac = (m > 10 * m.min()).mean()
    assert frac == pytest.approx(10**-1.35, rel=0.05)


def test_workload_king_w9():
    pos, vel, info = workloads.king(40000, 9.0, 5)
    r = np.linalg.norm(pos, axis=1)
    conc = math.log10(info["rt"] / info["r0"])
    assert conc == pytest.approx(2.12, abs=0.02)           # King (1966): W0 = 9 -> c = 2.12
    assert r.max() <= info["rt"] * (1 + 1e-9)
    # scaled to U = -1/2: virial T = 1/4
    assert 0.5 * (vel**2).sum(1).mean() == pytest.approx(0.25, rel=0.05)
    # much more concentrated than Plummer: 10 % Lagrangian radius is far smaller
    pp, _ = workloads.plummer(40000, 5)
    assert np.quantile(r, 0.1) < 0.5 * np.quantile(np.linalg.norm(pp, axis=1), 0.1)


def test_workload_configs_are_deterministic_and_fp32():
    a, b = workloads.config(1), workloads.config(1)
    assert a["pos"].dtype == np.float32 and a["mass"].dtype == np.float32
    assert np.array_equal(a["pos"], b["pos"])
    assert a["n"] == 4096 and a["r_in"] == pytest.approx(0.001, rel=1e-6)
    c2 = workloads.config(2, n=1024)
    assert c2["r_search"] == pytest.approx(c2["r_out"] + 3 / math.sqrt(2) / 256, rel=1e-6)
    c3 = workloads.config(3, n=4096)
    assert c3["mass"].sum() == pytest.approx(1.0, rel=1e-5) and c3["mass"].max() / c3["mass"].min() > 50
