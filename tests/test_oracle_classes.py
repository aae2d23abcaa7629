"""Pins of oracle part O8: per-pair-class cutoffs (section 3.2.2.1: r_cut,FS-FS, r_cut,BH-FS, unsplit BH-BH).

Each pin checks the class-aware functions against something other than themselves: formulas written out here with
numpy and the single-class K, W (pinned by test_oracle_cutoff.py), closed forms, python loops, finite differences,
and the reduction to the single-class oracle parts O2 / O3 / O6 / O4.
"""
import numpy as np
import pytest

EPS, R_IN, R_OUT, H = 1e-3, 0.01, 0.1, 0.12
R_IN_BF, R_OUT_BF, H_BF = 0.04, 0.4, 0.45
EPS_BB = 0.0


def _system(n=60, nbh=3, seed=5):
    rng = np.random.default_rng(seed)
    q = rng.uniform(-0.5, 0.5, (n, 3))
    q[1] = q[0] + [0.004, 0.0, 0.0]          # FS-FS pair inside r_in
    q[3] = q[2] + [0.05, 0.0, 0.0]           # FS-FS pair inside the transition
    m = rng.uniform(0.5, 1.5, n) / n
    cls = np.zeros(n, dtype=np.uint8)
    cls[-nbh:] = 1
    m[-nbh:] *= 20
    q[4] = q[-1] + [0.02, 0.01, 0.0]         # FS inside r_in,BF of a BH
    q[5] = q[-1] + [0.0, 0.2, 0.05]          # FS in the BH-FS transition
    v = rng.normal(0, 1, (n, 3))
    return m, q, v, cls


def _tab(oracle):
    return oracle.pair_table(EPS, R_IN, R_OUT, H, R_IN_BF, R_OUT_BF, H_BF, eps_bb=EPS_BB)


def _kind_params(ci, cj):
    k = int(ci) + int(cj)
    return [(EPS, R_IN, R_OUT, H), (EPS, R_IN_BF, R_OUT_BF, H_BF), (EPS_BB, np.inf, np.inf, np.inf)][k]


def _KW(oracle, s, r_in, r_out):
    if np.isinf(r_out):
        return 0.0, 0.0
    if s >= r_out:
        return 1.0, 1.0
    return oracle.pair_weights(s, r_in, r_out)


def _loops(oracle, m, q, cls):
    """soft and hard sums, lists: plain python loops over pairs with the kind's own numbers"""
    n = len(m)
    a_s, a_h, p_s, p_h = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros(n), np.zeros(n)
    lists = [[] for _ in range(n)]
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            eps, r_in, r_out, h = _kind_params(cls[i], cls[j])
            d = q[i] - q[j]
            s = np.sqrt(d @ d + eps * eps)
            K, W = _KW(oracle, s, r_in, r_out)
            a_s[i] -= m[j] * K * d / s ** 3
            a_h[i] -= m[j] * (1 - K) * d / s ** 3
            p_s[i] -= m[j] * W / s
            p_h[i] -= m[j] * (1 - W) / s
            if np.isinf(r_out) or s < h:
                lists[i].append(j)
    return a_s, p_s, a_h, p_h, lists


def test_C1_direct_sums_and_lists_equal_python_loops_with_the_kinds_own_numbers(oracle):
    m, q, v, cls = _system()
    tab = _tab(oracle)
    a_s, p_s, a_h, p_h = oracle.direct_classes(m, q, cls, tab, hard=True)
    ra_s, rp_s, ra_h, rp_h, lists = _loops(oracle, m, q, cls)
    np.testing.assert_allclose(a_s, ra_s, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(a_h, ra_h, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(p_s, rp_s, rtol=1e-12)
    np.testing.assert_allclose(p_h, rp_h, rtol=1e-11, atol=1e-13)
    off, lst, band = oracle.neighbours_classes(q, cls, tab)
    assert len(band) == 0
    assert [lst[off[i]:off[i + 1]].tolist() for i in range(len(m))] == lists
    bh = np.flatnonzero(cls == 1)
    for i in bh:                                   # black holes always list each other (unsplit, L287)
        assert set(bh) - {i} <= set(lists[i])
    assert any(len(lists[i]) > 0 for i in np.flatnonzero(cls == 0))


def test_C2_soft_plus_hard_is_plain_newton_with_the_kinds_softening(oracle):
    m, q, v, cls = _system()
    a_s, p_s, a_h, p_h = oracle.direct_classes(m, q, cls, _tab(oracle), hard=True)
    n = len(m)
    for i in range(n):
        d = q[i] - np.delete(q, i, axis=0)
        eps = np.where((cls[i] == 1) & (np.delete(cls, i) == 1), EPS_BB, EPS)
        s2 = (d * d).sum(1) + eps ** 2
        mj = np.delete(m, i)
        np.testing.assert_allclose(a_s[i] + a_h[i], -(mj[:, None] * d / s2[:, None] ** 1.5).sum(0), rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(p_s[i] + p_h[i], -(mj / np.sqrt(s2)).sum(), rtol=1e-12)
    # the hard function over all pairs gives the same hard part
    a, j, p = oracle.hard_classes(m, q, v, cls, _tab(oracle))
    np.testing.assert_allclose(a, a_h, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(p, p_h, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("ci,cj", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_C3_two_body_closed_forms_per_kind(oracle, ci, cj):
    eps, r_in, r_out, h = _kind_params(ci, cj)
    m = np.array([0.7, 0.3])
    cls = np.array([ci, cj], dtype=np.uint8)
    tab = _tab(oracle)
    top = 1.0 if np.isinf(r_out) else 2.0 * r_out
    for r in np.linspace(0.003, top, 41):
        q = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
        s = np.sqrt(r * r + eps * eps)
        K, W = _KW(oracle, s, r_in, r_out)
        a_s, p_s, a_h, p_h = oracle.direct_classes(m, q, cls, tab, hard=True)
        assert a_s[0, 0] == pytest.approx(m[1] * K * r / s ** 3, rel=1e-12, abs=1e-300)
        assert a_h[0, 0] == pytest.approx(m[1] * (1 - K) * r / s ** 3, rel=1e-12, abs=1e-300)
        assert p_s[1] == pytest.approx(-m[0] * W / s, rel=1e-12, abs=1e-300)
        off, lst, _ = oracle.neighbours_classes(q, cls, tab, band=0.0)
        assert (off[-1] == 2) == (np.isinf(r_out) or s < h)
    if ci + cj == 2:                               # unsplit: no soft force at any distance, all of it hard, unsoftened
        assert np.all(a_s == 0) and np.all(p_s == 0)
        assert a_h[0, 0] == pytest.approx(m[1] / top ** 2, rel=1e-12)


def test_C4_momentum_is_conserved_across_classes(oracle):
    m, q, v, cls = _system(n=80, nbh=4, seed=11)
    a_s, p_s, a_h, p_h = oracle.direct_classes(m, q, cls, _tab(oracle), hard=True)
    scale = (m[:, None] * np.abs(a_s)).sum()
    assert np.abs((m[:, None] * a_s).sum(0)).max() < 1e-13 * scale
    assert np.abs((m[:, None] * a_h).sum(0)).max() < 1e-13 * (m[:, None] * np.abs(a_h)).sum()


def test_C5_soft_acceleration_is_minus_the_gradient_of_the_soft_energy(oracle):
    m, q, v, cls = _system(n=40, nbh=2, seed=3)
    tab = _tab(oracle)

    def energy(qq):
        _, p = oracle.direct_classes(m, qq, cls, tab)
        return 0.5 * (m * p).sum()

    a, _ = oracle.direct_classes(m, q, cls, tab)
    for i in (0, 4, 5, len(m) - 1, len(m) - 2):
        for c in range(3):
            d = 1e-6
            qp, qm = q.copy(), q.copy()
            qp[i, c] += d
            qm[i, c] -= d
            g = (energy(qp) - energy(qm)) / (2 * d)
            assert a[i, c] == pytest.approx(-g / m[i], rel=2e-6, abs=1e-7 * np.abs(a[i]).max())


def test_C6_jerk_is_the_time_derivative_of_the_hard_acceleration(oracle):
    m, q, v, cls = _system(n=40, nbh=3, seed=8)
    tab = _tab(oracle)
    a, j, p = oracle.hard_classes(m, q, v, cls, tab)
    dt = 1e-6
    ap, _, _ = oracle.hard_classes(m, q + dt * v, v, cls, tab)
    am, _, _ = oracle.hard_classes(m, q - dt * v, v, cls, tab)
    fd = (ap - am) / (2 * dt)
    busy = np.abs(a).sum(1) > 0
    assert busy.sum() >= 6
    np.testing.assert_allclose(j[busy], fd[busy], rtol=2e-5, atol=1e-6 * np.abs(j).max())


def test_C7_one_class_reduces_to_the_single_class_oracle_parts(oracle):
    m, q, v, cls = _system()
    cls0 = np.zeros_like(cls)
    tab = _tab(oracle)
    a_s, p_s, a_h, p_h = oracle.direct_classes(m, q, cls0, tab, hard=True)
    b_s, q_s, b_h, q_h = oracle.direct(m, q, EPS, R_IN, R_OUT, hard=True)
    assert np.array_equal(a_s, b_s) and np.array_equal(p_s, q_s) and np.array_equal(a_h, b_h) and np.array_equal(p_h, q_h)
    off, lst, _ = oracle.neighbours_classes(q, cls0, tab)
    off0, lst0, _ = oracle.neighbours(q, EPS, H)
    assert np.array_equal(off, off0) and np.array_equal(lst, lst0)
    a, j, p = oracle.hard_classes(m, q, v, cls0, tab)
    a0, j0, p0 = oracle.hard(m, q, v, EPS, R_IN, R_OUT)
    assert np.array_equal(a, a0) and np.array_equal(j, j0) and np.array_equal(p, p0)


def test_C8_tree_walk_with_classes(oracle):
    from paper_1506_04553_b200 import workloads

    cfg = workloads.config(6, n=3000)
    m, q, cls = cfg["mass"].astype(np.float64), cfg["pos"].astype(np.float64), cfg["classes"]
    cp = cfg["class_params"]
    tab = oracle.pair_table(cfg["eps"], cfg["r_in"], cfg["r_out"], cfg["r_search"], cp["r_in_bf"], cp["r_out_bf"],
                            cp["r_search_bf"], eps_bb=cp["eps_bb"])
    a, p = oracle.direct_classes(m, q, cls, tab)
    off, lst, band = oracle.neighbours_classes(q, cls, tab)
    assert len(band) == 0
    n = len(m)
    assert off[n] - off[n - 1] >= 1 and (n - 2) in lst[off[n - 1]:off[n]].tolist()       # the holes list each other
    assert np.diff(off)[-2:].sum() >= 3                                                 # and field stars within h_BF = 1/32 + buffer
    tree = oracle.Tree(m, q, nleaf=16)
    stride = int(np.diff(off).max()) + 1
    # theta = 0: the walk IS the direct sum
    w0 = tree.walk_classes(cls, tab, 0.0, nbr_stride=stride)
    np.testing.assert_allclose(w0["acc"], a, rtol=1e-11, atol=1e-12 * np.abs(a).max())
    np.testing.assert_allclose(w0["pot"], p, rtol=1e-12)
    errs = []
    for theta in (0.8, 0.4):
        w = tree.walk_classes(cls, tab, theta, nbr_stride=stride)
        # lists through the walk are the exact ones whatever theta (clause 3 of R-MAC with the kind's own h)
        assert np.array_equal(w["nbr_count"], np.diff(off))
        for i in list(range(0, n, 97)) + [n - 2, n - 1]:
            assert w["nbr"][i, :w["nbr_count"][i]].tolist() == lst[off[i]:off[i + 1]].tolist()
        err = np.linalg.norm(w["acc"] - a, axis=1) / np.linalg.norm(a, axis=1)
        errs.append(np.median(err))
        assert np.percentile(err, 99) < (1e-2 if theta <= 0.4 else 5e-2) and w["n_pc"].sum() > 0
        # a black-hole target never takes a cell that holds the other black hole: its soft force has no BH-BH part
        for i in (n - 2, n - 1):
            assert err[i] < 1e-2
    assert errs[1] < errs[0]
    # all classes 0 with a one-kind table = the single-class walk, bit for bit
    cls0 = np.zeros_like(cls)
    w1 = tree.walk_classes(cls0, tab, 0.4)
    w2 = tree.walk(cfg["eps"], 0.4, cfg["r_in"], cfg["r_out"], cfg["r_search"])
    assert np.array_equal(w1["acc"], w2["acc"]) and np.array_equal(w1["pot"], w2["pot"]) and np.array_equal(w1["n_pc"], w2["n_pc"])
    # a box that holds a black hole opens every cell that holds the other one and everything within h_BF
    i = 10
    box = np.concatenate([np.minimum(q[i], q[n - 1]), np.maximum(q[i], q[n - 1])])[None, :]
    wb = tree.walk_classes(cls, tab, 0.4, subset=[i], box=box, box_mask=[3])
    wp = tree.walk_classes(cls, tab, 0.4, subset=[i])
    assert wb["n_pp"][0] > wp["n_pp"][0]
    assert np.linalg.norm(wb["acc"][0] - a[i]) <= np.linalg.norm(wp["acc"][0] - a[i]) * 1.05 + 1e-12


# ---- O7 with classes: the Hermite part of the SMBH runs (L287: eta_FS = 0.1, eta_BH = 0.03, BH-BH pure Hermite) ----------

def _hard_energy(oracle, m, q, v, cls, tab):
    _, _, p = oracle.hard_classes(m, q, v, cls, tab)
    return 0.5 * (m * (v * v).sum(1)).sum() + 0.5 * (m * p).sum()


def test_C9_hermite_with_one_class_is_the_single_class_integrator_bit_for_bit(oracle):
    rng = np.random.default_rng(21)
    n = 40
    q = rng.uniform(-0.15, 0.15, (n, 3))
    v = rng.normal(0, 0.3, (n, 3))
    m = rng.uniform(0.5, 1.5, n) / n
    cls = np.zeros(n, dtype=np.uint8)
    tab = _tab(oracle)
    off, lst, _ = oracle.neighbours(q, EPS, H)
    assert off[-1] > 20
    T, a0 = 1.0 / 64, 0.1 * m.mean() / R_OUT ** 2
    q1, v1, i1 = oracle.hermite(m, q, v, EPS, R_IN, R_OUT, off, lst, T, eta=0.1, eta_s=0.01, a0=a0)
    q2, v2, i2 = oracle.hermite_classes(m, q, v, cls, tab, off, lst, T, eta=(0.1, 0.1), eta_s=(0.01, 0.01), a0=(a0, a0))
    assert np.array_equal(q1, q2) and np.array_equal(v1, v2)
    assert i1["blocks"] == i2["blocks"] and np.array_equal(i1["nstep"], i2["nstep"])


def test_C10_two_black_holes_far_apart_are_a_pure_hermite_kepler_orbit(oracle):
    """Kind 2 is not split: whatever their distance the two holes are in each other's list and feel the whole unsoftened
    Newtonian force.  Circular orbit of separation 1 (32 times r_cut,BH-FS): the closed form, at fourth order in eta."""
    m = np.array([0.01, 0.01])
    M, r = m.sum(), 1.0
    w = np.sqrt(M / r ** 3)
    q = np.array([[0.5, 0, 0], [-0.5, 0, 0]], dtype=np.float64)
    v = np.array([[0, 0.5 * r * w, 0], [0, -0.5 * r * w, 0]])
    cls = np.array([1, 1], dtype=np.uint8)
    tab = _tab(oracle)
    off, lst, _ = oracle.neighbours_classes(q, cls, tab)
    assert lst.tolist() == [1, 0]
    T = 0.3 * 2 * np.pi / w
    exact = 0.5 * r * np.array([np.cos(w * T), np.sin(w * T), 0.0])
    errs = []
    for eta in (0.2, 0.1, 0.05):
        q1, v1, info = oracle.hermite_classes(m, q, v, cls, tab, off, lst, T, log2_div=3, eta=(0.1, eta), eta_s=(0.01, 0.1 * eta))
        errs.append(np.linalg.norm(q1[0] - exact))
        assert np.allclose(q1[0], -q1[1], atol=1e-14)
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1e-6
    assert errs[0] / errs[2] > 30                                  # fourth order: about 2^4 per halving of eta (block steps quantise it)
    # the same two bodies as field stars: far beyond r_cut, empty lists, a plain drift
    cls0 = np.zeros(2, dtype=np.uint8)
    off0, lst0, _ = oracle.neighbours_classes(q, cls0, tab)
    assert off0[-1] == 0
    q0, v0, _ = oracle.hermite_classes(m, q, v, cls0, tab, off0, lst0, T)
    assert np.array_equal(q0, q + T * v) and np.array_equal(v0, v)


def test_C11_hard_energy_is_conserved_across_kinds_and_eta_is_per_class(oracle):
    """A hole with two field stars inside r_cut,BH-FS (one inside r_in,BH-FS), a close pair of field stars, a second hole far
    away: H_hard = kinetic energy + hard potential of O8 is conserved over a soft step, better with smaller eta; the
    hole's step count follows eta_BH, the stars' follow eta_FS."""
    m = np.array([0.02, 1e-3, 1e-3, 1e-3, 1e-3, 0.02])
    q = np.array([[0, 0, 0], [0.03, 0, 0], [0, 0.2, 0.05], [0.6, 0.6, 0.0], [0.6, 0.605, 0.0], [-0.7, 0.1, 0.0]], dtype=np.float64)
    v = np.array([[0, 0, 0], [0, 0.8, 0], [0.25, 0, 0], [0, 0, 0.02], [0.3, 0, -0.02], [0, -0.1, 0]], dtype=np.float64)
    cls = np.array([1, 0, 0, 0, 0, 1], dtype=np.uint8)
    tab = _tab(oracle)
    off, lst, band = oracle.neighbours_classes(q, cls, tab)
    assert len(band) == 0 and 5 in lst[off[0]:off[1]].tolist() and 4 in lst[off[3]:off[4]].tolist()
    e0 = _hard_energy(oracle, m, q, v, cls, tab)
    T = 0.02
    drift = []
    for eta in (0.2, 0.05):
        q1, v1, info = oracle.hermite_classes(m, q, v, cls, tab, off, lst, T, eta=(eta, eta), eta_s=(0.1 * eta, 0.1 * eta),
                                              a0=(0.1 * 1e-3 / R_OUT ** 2, 0.1 * 0.02 / R_OUT_BF ** 2))
        drift.append(abs(_hard_energy(oracle, m, q1, v1, cls, tab) - e0) / abs(e0))
    assert drift[1] < drift[0] and drift[1] < 1e-7
    a0 = (0.1 * 1e-3 / R_OUT ** 2, 0.1 * 0.02 / R_OUT_BF ** 2)
    _, _, ia = oracle.hermite_classes(m, q, v, cls, tab, off, lst, T, eta=(0.1, 0.1), eta_s=(0.01, 0.01), a0=a0)
    _, _, ib = oracle.hermite_classes(m, q, v, cls, tab, off, lst, T, eta=(0.1, 0.03), eta_s=(0.01, 0.003), a0=a0)
    assert ib["nstep"][0] > ia["nstep"][0] and ib["nstep"][5] >= ia["nstep"][5]       # the holes step more finely
    assert np.array_equal(ib["nstep"][3:5], ia["nstep"][3:5])                          # the far pair of stars does not care
