"""Pins for the oracle's direct sum (O2) and neighbour sets (O3).

P6   a_i = -(1/m_i) dH_soft/dq_i by central differences      Eq. 6, 8 L55-65
P7   soft + hard = plain softened Newtonian; r_cut <= eps     Eq. 4-7
P8   two-body closed form swept over s                        Eq. 8
P9   sum_i m_i a_i = 0                                        Eq. 8 (K depends on s only)
P10  Plummer potential energy -> -1/2 (1 - sum m_i^2)         L163 (E = -1/4 => U = -1/2)
P11  neighbour symmetry, brute force vs tiny python loop,     L138-140; Eq. 22
     sweep == brute force, expected mean list length
"""
import math

import numpy as np
import pytest

from paper_1506_04553_b200 import workloads


def _cluster(n, seed, scale):
    """Random bodies with pair separations inside, across and outside [r_in, r_cut]."""
    rng = np.random.default_rng(seed)
    pos = rng.normal(0.0, scale, (n, 3))
    for k, sep in enumerate((0.004, 0.009, 0.015, 0.03, 0.06)):   # explicit close companions
        pos[2 * k + 1] = pos[2 * k] + sep * np.array([0.6, -0.48, 0.64])
    mass = rng.uniform(0.5, 1.5, n) / n
    return mass, pos


def test_p6_acc_is_gradient_of_Hsoft(oracle):
    r_in, r_out, eps = 0.02, 0.2, 0.013
    mass, pos = _cluster(64, 1, 0.15)
    s = np.sqrt(((pos[:, None] - pos[None]) ** 2).sum(-1) + eps**2)[np.triu_indices(64, 1)]
    assert (s < r_in).any() and ((s > r_in) & (s < r_out)).sum() > 50 and (s > r_out).sum() > 50
    acc, _ = oracle.direct(mass, pos, eps, r_in, r_out)

    def H(p):
        _, phi = oracle.direct(mass, p, eps, r_in, r_out)
        return 0.5 * np.sum(mass * phi)

    d = 1e-6
    for i in (0, 1, 3, 4, 7, 31, 63):
        for ax in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[i, ax] += d
            pm[i, ax] -= d
            grad = (H(pp) - H(pm)) / (2 * d)
            assert acc[i, ax] == pytest.approx(-grad / mass[i], rel=2e-7, abs=1e-9)


def test_p7_soft_plus_hard_is_newton(oracle):
    r_in, r_out, eps = 0.02, 0.2, 0.013
    mass, pos = _cluster(200, 2, 0.15)
    a_s, p_s, a_h, p_h = oracle.direct(mass, pos, eps, r_in, r_out, hard=True)
    d = pos[:, None] - pos[None]
    s2 = (d**2).sum(-1) + eps**2
    np.fill_diagonal(s2, np.inf)
    a_n = -(mass[None, :, None] * d / s2[..., None] ** 1.5).sum(1)
    p_n = -(mass[None] / np.sqrt(s2)).sum(1)
    np.testing.assert_allclose(a_s + a_h, a_n, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(p_s + p_h, p_n, rtol=1e-12)
    assert np.abs(a_h).max() > 1e-3  # the split is not trivial for this cluster


def test_p7_rcut_below_eps_is_plain_newton(oracle):
    mass, pos = _cluster(100, 3, 0.1)
    eps = 0.05
    a_s, p_s, a_h, p_h = oracle.direct(mass, pos, eps, 0.001, 0.01, hard=True)
    assert np.all(a_h == 0.0) and np.all(p_h == 0.0)
    d = pos[:, None] - pos[None]
    s2 = (d**2).sum(-1) + eps**2
    np.fill_diagonal(s2, np.inf)
    np.testing.assert_allclose(p_s, -(mass[None] / np.sqrt(s2)).sum(1), rtol=1e-13)


def test_p8_two_body_closed_form(oracle):
    r_in, r_out, eps = 0.1, 1.0, 0.05
    m = np.array([0.3, 0.7])
    u = np.array([1.0, 2.0, -2.0]) / 3.0
    for sep in np.linspace(1e-3, 2.0, 41):
        pos = np.stack([np.zeros(3), sep * u])
        acc, pot = oracle.direct(m, pos, eps, r_in, r_out)
        s = math.sqrt(sep**2 + eps**2)
        k, w = oracle.pair_weights(s, r_in, r_out)
        # a_1 = -m_2 K(s) (q_1 - q_2)/s^3, q_1 - q_2 = -sep u
        np.testing.assert_allclose(acc[0], m[1] * k * sep * u / s**3, rtol=1e-13, atol=1e-16)
        np.testing.assert_allclose(acc[1], -m[0] * k * sep * u / s**3, rtol=1e-13, atol=1e-16)
        assert pot[0] == pytest.approx(-m[1] * w / s, rel=1e-13)
    # end conditions of north_star, in the form the equations allow (reading A3):
    acc, _ = oracle.direct(m, np.stack([np.zeros(3), 0.08 * u]), eps, r_in, r_out)  # s < r_in
    assert np.all(acc == 0.0)


def test_p9_momentum_conservation(oracle):
    c = workloads.config(1, n=1024)
    m, q = c["mass"].astype(np.float64), c["pos"].astype(np.float64)
    acc, _ = oracle.direct(m, q, c["eps"], 0.01, 0.1)
    f = (m[:, None] * acc).sum(0)
    assert np.abs(f).max() < 1e-13 * np.abs(m[:, None] * acc).sum()


def test_p10_plummer_potential_energy(oracle):
    n = 8192
    pos, _ = workloads.plummer(n, 12345)
    m = np.full(n, 1.0 / n)
    eps = 1e-4
    _, phi = oracle.direct(m, pos, eps, 0.1 * eps * 0.5, eps * 0.5)  # r_cut <= eps: cutoff disabled
    u = 0.5 * np.sum(m * phi)
    expect = -0.5 * (1.0 - np.sum(m * m))
    # sampling noise ~ 1/sqrt(n) * O(1); truncation at 20a removes ~0.4 % of the mass at large r
    assert u == pytest.approx(expect, abs=3.0 / math.sqrt(n))
    assert u < -0.45


def test_p11_neighbours_vs_python_loop_and_symmetry(oracle):
    rng = np.random.default_rng(5)
    pos = rng.uniform(0, 1, (300, 3))
    eps, h = 0.03, 0.15
    off, lst, _ = oracle.neighbours(pos, eps, h)
    sets = [set(lst[off[i]:off[i + 1]].tolist()) for i in range(300)]
    for i in range(300):
        want = {j for j in range(300) if j != i and math.sqrt(((pos[i] - pos[j]) ** 2).sum() + eps**2) < h}
        assert sets[i] == want
        assert list(lst[off[i]:off[i + 1]]) == sorted(want)
    assert all(i in sets[j] for i in range(300) for j in sets[i])
    assert off[-1] % 2 == 0
    # plain-distance variant (reading A4's alternative) is a superset
    off2, lst2, _ = oracle.neighbours(pos, eps, h, plain=True)
    assert off2[-1] > off[-1]


def test_p11_subset_and_band(oracle):
    rng = np.random.default_rng(6)
    pos = rng.uniform(0, 1, (400, 3))
    pos[1] = pos[0] + np.array([0.1 * (1 + 2e-7), 0.0, 0.0])   # inside the 1e-6 band around h = 0.1
    sub = np.array([0, 17, 250])
    off, lst, band = oracle.neighbours(pos, 0.0, 0.1, subset=sub)
    off_all, lst_all, _ = oracle.neighbours(pos, 0.0, 0.1)
    for k, i in enumerate(sub):
        assert list(lst[off[k]:off[k + 1]]) == list(lst_all[off_all[i]:off_all[i + 1]])
    assert [0, 1] in band.tolist()


def test_p11_sweep_equals_brute_force(oracle):
    c = workloads.config(1, n=4096)
    q = c["pos"].astype(np.float64)
    for h in (0.012, 0.12):
        off, lst, _ = oracle.neighbours(q, c["eps"], h)
        off2, lst2 = oracle.neighbours_sweep(q, c["eps"], h)
        assert np.array_equal(off, off2) and np.array_equal(lst, lst2)


def test_p11_expected_list_length_plummer(oracle):
    # Eq. 22 (L202): N_ngh,i ~ (4 pi/3) h^3 n_i; averaged over a Plummer sphere
    # <n> = N int rho^2 dV / M^2 = N * 3/(4 pi a^3) * (pi/ (32/ (3*pi)))... evaluated numerically below
    n, h = 16384, 0.05
    pos, _ = workloads.plummer(n, 99)
    a = workloads.PLUMMER_A
    r = np.linspace(0, 40 * a, 400001)
    rho = 3 / (4 * math.pi * a**3) * (1 + (r / a) ** 2) ** -2.5
    mean_density = n * np.trapezoid(rho * rho * 4 * math.pi * r * r, r)
    expect = 4 * math.pi / 3 * h**3 * mean_density
    off, _ = oracle.neighbours_sweep(pos, 0.0, h)
    got = off[-1] / n
    assert got == pytest.approx(expect, rel=0.08)   # finite-h smoothing lowers it by a few %
