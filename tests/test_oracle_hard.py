"""Pins of the oracle's hard-force part O6 (Eq. 7, Eq. 5), against things
other than itself: finite differences, the plain softened Newtonian force, a closed two-body form."""
import numpy as np
import pytest

from paper_1506_04553_b200 import workloads


def _case(n=96, seed=5):
    rng = np.random.default_rng(seed)
    q = rng.uniform(-1.0, 1.0, (n, 3)) * 0.05          # many pairs inside, across and outside [r_in, r_out]
    v = rng.normal(size=(n, 3))
    m = rng.uniform(0.5, 1.5, n) / n
    return m, q, v, 1e-3, 0.004, 0.04                   # eps, r_in, r_out


def test_h1_dKdx_is_the_derivative_of_K(oracle):
    for x in np.linspace(0.02, 0.98, 25):
        fd = (oracle.K(x + 1e-6) - oracle.K(x - 1e-6)) / 2e-6
        assert oracle.dKdx(x) == pytest.approx(fd, rel=1e-7, abs=2e-8)      # K near x = 1 cancels from terms of size 84
        expanded = -140.0 * x ** 6 + 420.0 * x ** 5 - 420.0 * x ** 4 + 140.0 * x ** 3      # term-by-term derivative of Eq. 12
        assert oracle.dKdx(x) == pytest.approx(expanded, rel=1e-9, abs=1e-12)
    assert oracle.dKdx(-0.1) == 0.0 and oracle.dKdx(0.0) == 0.0 and oracle.dKdx(1.0) == 0.0 and oracle.dKdx(1.5) == 0.0


def test_h2_hard_acceleration_and_potential_complete_the_soft_ones_to_plain_newton(oracle):
    m, q, v, eps, r_in, r_out = _case()
    a_h, j_h, p_h = oracle.hard(m, q, v, eps, r_in, r_out)
    a_s, p_s, a_h2, p_h2 = oracle.direct(m, q, eps, r_in, r_out, hard=True)
    assert np.allclose(a_h, a_h2, rtol=1e-13, atol=1e-16) and np.allclose(p_h, p_h2, rtol=1e-13, atol=1e-16)
    # plain softened Newton, written out here
    d = q[:, None, :] - q[None, :, :]
    s2 = (d ** 2).sum(-1) + eps ** 2
    np.fill_diagonal(s2, 1.0)
    w = m[None, :] / s2 ** 1.5
    np.fill_diagonal(w, 0.0)
    a_n = -(w[:, :, None] * d).sum(1)
    assert np.allclose(a_s + a_h, a_n, rtol=1e-11, atol=1e-14)
    assert np.abs(a_h).max() > 0 and np.abs(a_s).max() > 0


def test_h3_jerk_is_the_time_derivative_of_the_hard_acceleration(oracle):
    m, q, v, eps, r_in, r_out = _case()
    _, jerk, _ = oracle.hard(m, q, v, eps, r_in, r_out)
    dt = 1e-6
    ap, _, _ = oracle.hard(m, q + dt * v, v, eps, r_in, r_out)
    am, _, _ = oracle.hard(m, q - dt * v, v, eps, r_in, r_out)
    fd = (ap - am) / (2 * dt)
    scale = np.abs(jerk).max()
    assert scale > 0
    assert np.abs(jerk - fd).max() <= 1e-6 * scale


def test_h4_hard_acceleration_is_minus_the_gradient_of_the_hard_potential_energy(oracle):
    m, q, v, eps, r_in, r_out = _case(n=40, seed=9)

    def u(qq):                                           # potential part of H_hard (Eq. 5): 1/2 sum m_i phi_i
        return 0.5 * np.sum(m * oracle.hard(m, qq, v, eps, r_in, r_out)[2])

    a, _, _ = oracle.hard(m, q, v, eps, r_in, r_out)
    h = 1e-7
    for i, c in [(0, 0), (7, 1), (23, 2), (39, 0)]:
        qp, qm = q.copy(), q.copy()
        qp[i, c] += h
        qm[i, c] -= h
        fd = -(u(qp) - u(qm)) / (2 * h) / m[i]
        assert a[i, c] == pytest.approx(fd, rel=2e-6, abs=1e-9 * np.abs(a).max())


def test_h5_two_bodies_closed_form_and_no_hard_force_beyond_r_out(oracle):
    eps, r_in, r_out = 0.0, 0.01, 0.1
    m = np.array([0.3, 0.7])
    for r in [0.005, 0.02, 0.05, 0.09, 0.1, 0.15]:
        q = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
        v = np.array([[0.0, 0.0, 0.0], [0.2, 0.1, 0.0]])
        a, j, p = oracle.hard(m, q, v, eps, r_in, r_out)
        K, W = (1.0, 1.0) if r >= r_out else oracle.pair_weights(r, r_in, r_out)
        assert a[0, 0] == pytest.approx(m[1] * (1.0 - K) / r ** 2, rel=1e-12, abs=1e-300)
        assert p[0] == pytest.approx(-m[1] * (1.0 - W) / r, rel=1e-12, abs=1e-300)
        if r >= r_out:
            assert np.all(a == 0) and np.all(j == 0) and np.all(p == 0)
        if r <= r_in:                                    # plain Newton inside r_in: a = m q / r^3, jerk = m (v/r^3 - 3 (q.v) q / r^5)
            qv = r * 0.2
            assert j[0, 0] == pytest.approx(m[1] * (0.2 / r ** 3 - 3 * qv * r / r ** 5), rel=1e-12)
            assert j[0, 1] == pytest.approx(m[1] * 0.1 / r ** 3, rel=1e-12)
