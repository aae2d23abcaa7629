"""Pins of the oracle's Hermite part O7 (procedure step 3 L147, Eq. 18-20), against
things other than itself: Kepler closed forms, conservation laws, fourth-order convergence, locality, exact drift."""
import numpy as np
import pytest


def _two_body(r, ecc=0.0, m1=0.6, m2=0.4):
    """Two bodies at apocentre of a Kepler orbit with semi-major axis r, centre of mass at rest at the origin."""
    M = m1 + m2
    ra = r * (1.0 + ecc)
    vrel = np.sqrt(M * (2.0 / ra - 1.0 / r))
    q = np.array([[ra * m2 / M, 0, 0], [-ra * m1 / M, 0, 0.0]])
    v = np.array([[0, vrel * m2 / M, 0], [0, -vrel * m1 / M, 0.0]])
    period = 2.0 * np.pi * np.sqrt(r ** 3 / M)
    return np.array([m1, m2]), q, v, period


PAIR = (np.array([0, 1, 2]), np.array([1, 0], dtype=np.int32))


def test_s1_circular_orbit_follows_the_closed_form_at_fourth_order(oracle):
    """Inside r_in the hard force is plain Newton (K = 0, Eq. 12 first branch): x(t) = R (cos wt, sin wt)."""
    r = 0.01
    m, q, v, period = _two_body(r)
    T = 0.3 * period
    w = 2.0 * np.pi / period
    exact = np.stack([np.linalg.norm(q, axis=1) * np.sign(q[:, 0]) * np.cos(w * T),
                      np.linalg.norm(q, axis=1) * np.sign(q[:, 0]) * np.sin(w * T), np.zeros(2)], axis=1)
    errs = []
    for eta in (0.2, 0.1, 0.05):
        q2, v2, info = oracle.hermite(m, q, v, 0.0, 1.0, 2.0, *PAIR, T, log2_div=2, eta=eta, eta_s=eta / 10)
        errs.append(np.abs(q2 - exact).max() / r)
        assert info["floor_hits"] == 0
    assert errs[2] < 2e-6
    assert errs[0] / errs[1] > 6.0 and errs[1] / errs[2] > 8.0         # step halves -> error / 16 (block quantisation blurs it)


def test_s2_eccentric_orbit_conserves_energy_and_angular_momentum(oracle):
    r, ecc = 0.01, 0.7
    m, q, v, period = _two_body(r, ecc)

    def invariants(q, v):
        d = np.linalg.norm(q[0] - q[1])
        e = 0.5 * np.sum(m * (v ** 2).sum(1)) - m[0] * m[1] / d
        lz = np.sum(m * (q[:, 0] * v[:, 1] - q[:, 1] * v[:, 0]))
        return e, lz

    e0, l0 = invariants(q, v)
    assert e0 == pytest.approx(-m[0] * m[1] / (2 * r), rel=1e-12)      # vis-viva: the setup itself
    de = []
    for eta in (0.1, 0.05):
        q2, v2, info = oracle.hermite(m, q, v, 0.0, 1.0, 2.0, *PAIR, period, log2_div=3, eta=eta, eta_s=eta / 10)
        e1, l1 = invariants(q2, v2)
        de.append(abs(e1 / e0 - 1.0))
        assert abs(l1 / l0 - 1.0) < 1e-6
        assert len(set(np.diff(np.sort(info["nstep"])))) == 1          # both bodies share every block here
        assert np.abs(q2 - q).max() < 0.02 * r                         # back at apocentre after one period
    assert de[0] < 1e-5 and de[1] < de[0] / 6.0
    # the step shrinks at pericentre: more steps than a circular orbit of the same period and eta needs
    mc, qc, vc, pc = _two_body(r)
    _, _, ic = oracle.hermite(mc, qc, vc, 0.0, 1.0, 2.0, *PAIR, pc, log2_div=3, eta=0.05, eta_s=0.005)
    assert info["nstep"][0] > 1.5 * ic["nstep"][0]


def test_s3_particles_with_empty_lists_drift(oracle):
    rng = np.random.default_rng(3)
    n = 20
    q, v, m = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)), rng.uniform(1, 2, n)
    off = np.zeros(n + 1, dtype=np.int64)
    q2, v2, info = oracle.hermite(m, q, v, 1e-3, 0.01, 0.1, off, np.zeros(0, np.int32), 0.125)
    assert np.array_equal(q2, q + 0.125 * v) and np.array_equal(v2, v)
    assert info["blocks"] == 0 and not info["nstep"].any()


def test_s4_buffer_shell_pair_takes_the_maximum_step_and_moves_on_straight_lines(oracle):
    """Neighbours outside r_out but inside h feel no hard force (1 - K = 0): a = a1 = 0, Eq. 20 gives infinity,
    so each takes exactly 2^log2_div steps of Delta t_max and the Hermite result is the drift."""
    m = np.array([1.0, 1.0])
    q = np.array([[0.0, 0, 0], [0.15, 0, 0]])
    v = np.array([[0.0, 0.1, 0], [0, -0.1, 0.05]])
    q2, v2, info = oracle.hermite(m, q, v, 0.0, 0.01, 0.1, *PAIR, 0.25, log2_div=3)
    assert list(info["nstep"]) == [8, 8] and info["blocks"] == 8
    assert np.allclose(q2, q + 0.25 * v, rtol=0, atol=1e-16) and np.array_equal(v2, v)


def _cluster(seed, n=6, scale=0.02):
    rng = np.random.default_rng(seed)
    q = rng.normal(size=(n, 3)) * scale
    m = rng.uniform(0.5, 1.5, n) / n
    v = rng.normal(size=(n, 3)) * np.sqrt(m.sum() / scale) * 0.5
    return m, q, v


def _hard_energy(oracle, m, q, v, eps, r_in, r_out):
    """H_hard of Eq. 5 (L53): kinetic energy + 1/2 sum_i m_i phi_hard,i, phi from O6 (pinned in test_oracle_hard)."""
    return 0.5 * np.sum(m * (v ** 2).sum(1)) + 0.5 * np.sum(m * oracle.hard(m, q, v, eps, r_in, r_out)[2])


def test_s5_hard_hamiltonian_is_conserved_across_the_cutoff(oracle):
    """A small cluster whose separations span the changeover and r > r_out, several pairs crossing r_out during the
    step; all-to-all lists.  Delta t_max = T/32: a body outside every cutoff sphere has a = 0 and takes the maximum
    step, which must stay small against r_out / v (L152: a_0, Delta t_max)."""
    eps, r_in, r_out = 1e-4, 0.004, 0.04
    m, q, v = _cluster(11)
    v = 0.5 * v
    n = len(m)
    off = np.arange(n + 1, dtype=np.int64) * (n - 1)
    lst = np.concatenate([[j for j in range(n) if j != i] for i in range(n)]).astype(np.int32)
    d = np.linalg.norm(q[:, None] - q[None], axis=-1)[np.triu_indices(n, 1)]
    assert (d < r_out).any() and (d > r_out).any()
    e0 = _hard_energy(oracle, m, q, v, eps, r_in, r_out)
    T = 0.02
    errs = []
    for eta in (0.1, 0.05, 0.025):
        q2, v2, info = oracle.hermite(m, q, v, eps, r_in, r_out, off, lst, T, log2_div=5, eta=eta, eta_s=eta / 10,
                                      a0=0.1 * m.mean() / r_out ** 2)
        errs.append(abs(_hard_energy(oracle, m, q2, v2, eps, r_in, r_out) - e0) / abs(e0))
        assert info["floor_hits"] == 0
    d2 = np.linalg.norm(q2[:, None] - q2[None], axis=-1)[np.triu_indices(n, 1)]
    assert np.sum((d < r_out) != (d2 < r_out)) >= 3                    # pairs entered / left the cutoff sphere
    assert errs[0] < 1e-5 and errs[2] < errs[0] / 20.0


def test_s6_clusters_that_share_no_list_entry_do_not_see_each_other(oracle):
    """Locality: integrating two clusters together equals integrating each alone (block times are global, the
    arithmetic of a particle only involves its list)."""
    eps, r_in, r_out = 1e-4, 0.004, 0.04
    ma, qa, va = _cluster(21, n=4)
    mb, qb, vb = _cluster(22, n=5)
    qb = qb + np.array([10.0, 0, 0])

    def full(n):
        return (np.arange(n + 1, dtype=np.int64) * (n - 1),
                np.concatenate([[j for j in range(n) if j != i] for i in range(n)]).astype(np.int32))

    oa, la = full(4)
    ob, lb = full(5)
    m, q, v = np.concatenate([ma, mb]), np.concatenate([qa, qb]), np.concatenate([va, vb])
    off = np.concatenate([oa, oa[-1] + ob[1:]])
    lst = np.concatenate([la, lb + 4]).astype(np.int32)
    T, a0 = 0.01, 0.1 * 0.2 / r_out ** 2
    q2, v2, _ = oracle.hermite(m, q, v, eps, r_in, r_out, off, lst, T, a0=a0)
    qa2, va2, _ = oracle.hermite(ma, qa, va, eps, r_in, r_out, oa, la, T, a0=a0)
    qb2, vb2, _ = oracle.hermite(mb, qb, vb, eps, r_in, r_out, ob, lb, T, a0=a0)
    assert np.array_equal(q2[:4], qa2) and np.array_equal(v2[:4], va2)
    assert np.array_equal(q2[4:], qb2) and np.array_equal(v2[4:], vb2)


def test_s7_relabelling_the_particles_changes_nothing_but_rounding(oracle):
    eps, r_in, r_out = 1e-4, 0.004, 0.04
    m, q, v = _cluster(31, n=7)
    n = 7
    off = np.arange(n + 1, dtype=np.int64) * (n - 1)
    lst = np.concatenate([[j for j in range(n) if j != i] for i in range(n)]).astype(np.int32)
    a0 = 0.1 * m.mean() / r_out ** 2
    q2, v2, _ = oracle.hermite(m, q, v, eps, r_in, r_out, off, lst, 0.01, a0=a0)
    perm = np.random.default_rng(0).permutation(n)
    q3, v3, _ = oracle.hermite(m[perm], q[perm], v[perm], eps, r_in, r_out, off, lst, 0.01, a0=a0)
    assert np.allclose(q3, q2[perm], rtol=0, atol=1e-12) and np.allclose(v3, v2[perm], rtol=1e-9, atol=1e-9)


def test_s8_whole_scheme_conserves_the_total_energy_at_second_order_in_the_soft_step(oracle):
    """Steps 1-5 of L142-153 on a small Plummer-like cluster with the soft force by direct sum: the energy error is
    that of the leapfrog splitting, O(dt_soft^2) (L187: 'the error is dominated by the truncation error of the
    leapfrog integrator')."""
    rng = np.random.default_rng(8)
    n = 64
    q = rng.normal(size=(n, 3)) * 0.4
    v = rng.normal(size=(n, 3)) * 0.45
    m = np.full(n, 1.0 / n)
    eps, r_out = 4.0 / n * 0.1, 0.12
    r_in = 0.1 * r_out

    def energy(q, v):
        d = np.sqrt(((q[:, None] - q[None]) ** 2).sum(-1) + eps ** 2)
        iu = np.triu_indices(n, 1)
        return 0.5 * np.sum(m * (v ** 2).sum(1)) - np.sum((m[:, None] * m[None])[iu] / d[iu])

    e0 = energy(q, v)
    errs = []
    for nsteps in (32, 64, 128):
        T = 0.5 / nsteps
        h = r_out + 3.0 * 0.8 * T
        qq, vv = q.copy(), v.copy()
        a, _ = oracle.direct(m, qq, eps, r_in, r_out)
        off, lst, _ = oracle.neighbours(qq, eps, h)
        hermite_steps, worst = 0, 0.0
        for _ in range(nsteps):
            qq, vv, a, off, lst, info = oracle.p3t_step(m, qq, vv, a, off, lst, eps, r_in, r_out, h, T, eta=0.05,
                                                        eta_s=0.005, a0=0.1 * m[0] / r_out ** 2)
            hermite_steps += int(info["nstep"].sum())
            worst = max(worst, abs(energy(qq, vv) / e0 - 1.0))
        assert hermite_steps > 1000
        errs.append(worst)
    assert errs[2] < 1e-4
    assert errs[0] / errs[1] > 2.5 and errs[1] / errs[2] > 2.5         # second order: factor 4 per halving


def _ode_reference(oracle, m, q, v, T, accel):
    """Plain ODE solution x'' = accel(x) with scipy's DOP853 at rtol 1e-12 (an integrator that shares nothing with O7)."""
    from scipy.integrate import solve_ivp
    n = len(m)

    def rhs(t, y):
        x = y[: 3 * n].reshape(n, 3)
        return np.concatenate([y[3 * n:], accel(x).ravel()])

    sol = solve_ivp(rhs, (0.0, T), np.concatenate([q.ravel(), v.ravel()]), method="DOP853", rtol=1e-12, atol=1e-15)
    return sol.y[: 3 * n, -1].reshape(n, 3), sol.y[3 * n:, -1].reshape(n, 3)


def test_s9_hard_part_is_the_solution_of_the_hard_equations_of_motion(oracle):
    """Four bodies whose separations cross r_in and r_out, forces of Eq. 7 written out here with K from O1 (pinned in
    test_oracle_cutoff), integrated by DOP853: O7 converges to that solution at fourth order in eta."""
    eps, r_in, r_out = 1e-3, 0.01, 0.1
    m = np.array([0.4, 0.3, 0.2, 0.1])
    q = np.array([[0.0, 0, 0], [0.06, 0.01, 0], [-0.03, 0.07, 0.02], [0.02, -0.09, 0.05]])
    v = np.array([[0.0, 0.5, 0], [0.3, -1.0, 0.2], [0.8, 0.1, -0.3], [-0.9, 0.6, 0.1]])
    n = 4

    def accel(x):
        a = np.zeros_like(x)
        for i in range(n):
            for j in range(n):
                if i == j:
                    continue
                d = x[i] - x[j]
                s = np.sqrt(d @ d + eps * eps)
                xx = (s / r_out - r_in / r_out) / (1.0 - r_in / r_out)
                a[i] -= m[j] * (1.0 - oracle.K(xx)) * d / s ** 3
        return a

    T = 0.05
    qr, vr = _ode_reference(oracle, m, q, v, T, accel)
    off = np.arange(n + 1, dtype=np.int64) * (n - 1)
    lst = np.concatenate([[j for j in range(n) if j != i] for i in range(n)]).astype(np.int32)
    errs = []
    for eta in (0.2, 0.1, 0.05):
        q2, v2, info = oracle.hermite(m, q, v, eps, r_in, r_out, off, lst, T, log2_div=4, eta=eta, eta_s=eta / 10,
                                      a0=0.1 * m.mean() / r_out ** 2)
        errs.append(max(np.abs(q2 - qr).max() / np.abs(qr - q).max(), np.abs(v2 - vr).max() / np.abs(vr).max()))
    d0 = np.linalg.norm(q[:, None] - q[None], axis=-1)[np.triu_indices(n, 1)]
    d1 = np.linalg.norm(qr[:, None] - qr[None], axis=-1)[np.triu_indices(n, 1)]
    assert ((d0 < r_out) != (d1 < r_out)).any() or d1.min() < 0.5 * d0.min()       # the geometry did change
    assert errs[2] < 5e-6 and errs[0] > 5 * errs[1] > 25 * errs[2], errs          # observed 3.4e-4, 2.2e-5, 1.5e-6: factor 15 per halving


def test_s10_whole_scheme_converges_to_newtonian_motion_at_second_order(oracle):
    """Steps 1-5 (L142-153) against the DOP853 solution of the unsplit softened Newtonian equations: the splitting error
    is O(dt_soft^2) -- a wrong kick factor (a whole instead of half a kick, a missing second kick) breaks the order."""
    rng = np.random.default_rng(12)
    n = 12
    m = rng.uniform(0.5, 1.5, n) / n
    q = rng.normal(size=(n, 3)) * 0.15
    v = rng.normal(size=(n, 3)) * 0.8
    eps, r_out = 5e-3, 0.12
    r_in = 0.1 * r_out

    def accel(x):
        d = x[:, None, :] - x[None, :, :]
        s2 = (d ** 2).sum(-1) + eps ** 2
        np.fill_diagonal(s2, 1.0)
        w = m[None, :] / s2 ** 1.5
        np.fill_diagonal(w, 0.0)
        return -(w[:, :, None] * d).sum(1)

    Ttot = 0.1
    qr, vr = _ode_reference(oracle, m, q, v, Ttot, accel)
    errs = []
    for nsteps in (32, 64, 128):
        T = Ttot / nsteps
        h = r_out + 3.0 * T
        qq, vv = q.copy(), v.copy()
        a, _ = oracle.direct(m, qq, eps, r_in, r_out)
        off, lst, _ = oracle.neighbours(qq, eps, h)
        for _ in range(nsteps):
            qq, vv, a, off, lst, _info = oracle.p3t_step(m, qq, vv, a, off, lst, eps, r_in, r_out, h, T, log2_div=3, eta=0.02,
                                                         eta_s=0.002, a0=0.1 * m.mean() / r_out ** 2)
        errs.append(np.abs(qq - qr).max() / np.abs(qr - q).max())
    assert errs[2] < 5e-5, errs                                                   # observed 4.0e-4, 7.8e-5, 2.0e-5
    assert 2.5 < errs[0] / errs[1] < 7.0 and 2.5 < errs[1] / errs[2] < 7.0, errs
