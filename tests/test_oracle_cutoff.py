"""Pins for the oracle's cutoff functions K and W (O1).

P1  K end values, symmetry, flat derivatives        Eq. 12; L96-98
P2  K = 0 below r_in, K = W = 1 above r_cut         L59, L85, L102
P3  W - y dW/dy = K on (gamma, 1)                   Eq. 9 L68  (catches reading A1)
P4  W continuous at gamma and 1, W'(1) = 0, table   tests/golden/cutoff_gamma0p1.txt
P5  closed form == y [1 + int_y^1 K/t^2 dt]         Eq. 9 + W(1) = 1, scipy quadrature
"""
import os

import numpy as np
import pytest
from scipy.integrate import quad

GOLD = os.path.join(os.path.dirname(__file__), "golden", "cutoff_gamma0p1.txt")


def K_plain(x):
    """Eq. 12 retyped only for the quadrature integrand of P5 (the pin is the
    quadrature relation, not this polynomial)."""
    if x < 0:
        return 0.0
    if x >= 1:
        return 1.0
    return -20 * x**7 + 70 * x**6 - 84 * x**5 + 35 * x**4


def test_p1_K_values_and_symmetry(oracle):
    assert oracle.K(0.0) == 0.0
    assert oracle.K(1.0) == 1.0
    assert oracle.K(0.5) == pytest.approx(0.5, abs=1e-15)
    assert oracle.K(-0.3) == 0.0 and oracle.K(1.7) == 1.0
    x = np.linspace(0.0, 1.0, 201)
    k = oracle.K(x)
    np.testing.assert_allclose(k + oracle.K(1.0 - x), 1.0, atol=1e-14)
    assert np.all(np.diff(k) >= 0.0)  # monotone


def test_p1_K_three_flat_derivatives_at_both_ends(oracle):
    # lowest-order polynomial with derivatives up to third order zero at x = 0, 1 (L96-98):
    # K(d) = 35 d^4 + O(d^5) and 1 - K(1-d) = 35 d^4 + O(d^5)
    for d in (1e-2, 1e-3):
        assert oracle.K(d) / d**4 == pytest.approx(35.0, rel=3 * d)
        assert (1.0 - oracle.K(1.0 - d)) / d**4 == pytest.approx(35.0, rel=3 * d)


def test_p2_end_conditions_in_s(oracle):
    r_in, r_out = 0.001, 0.01
    for s in (1e-5, 5e-4, 0.001):
        k, w = oracle.pair_weights(s, r_in, r_out)
        assert k == 0.0
        # below r_in W/s is the constant C_in/r_cut: zero soft force (reading A3)
        assert w / s == pytest.approx(oracle.Cin(0.1) / r_out, rel=1e-13)
    for s in (0.01, 0.011, 1.0):
        assert oracle.pair_weights(s, r_in, r_out) == (1.0, 1.0)


@pytest.mark.parametrize("gamma", [0.1, 0.3, 0.5])
def test_p3_W_minus_y_dWdy_is_K(oracle, gamma):
    y = np.linspace(gamma + 1e-3, 1.0 - 1e-3, 97)
    h = 1e-5
    dW = (oracle.W(y + h, gamma) - oracle.W(y - h, gamma)) / (2 * h)
    lhs = oracle.W(y, gamma) - y * dW
    x = (y - gamma) / (1 - gamma)
    # the closed form cancels from terms of size ~57 (gamma=0.1) to ~1.2e4 (gamma=0.5);
    # divided by 2h that rounding shows up as 1e-9 .. 2e-7 in the difference quotient
    atol = {0.1: 2e-8, 0.3: 1e-7, 0.5: 1e-6}[gamma]
    np.testing.assert_allclose(lhs, oracle.K(x), atol=atol)


def test_p3_extracted_eq17_sign_is_rejected(oracle):
    # Eq. 17 exactly as extracted (denominator (1-gamma)^7) flips G's sign: then
    # W - y W' = -K.  Shows the test above discriminates between the two readings.
    g, y, h = 0.1, 0.5, 1e-5

    def W_bad(yy):
        return -oracle.G(yy, g) + (1.0 + oracle.G(1.0, g)) * yy

    lhs = W_bad(y) - y * (W_bad(y + h) - W_bad(y - h)) / (2 * h)
    assert lhs == pytest.approx(-float(oracle.K((y - g) / (1 - g))), abs=1e-7)


@pytest.mark.parametrize("gamma", [0.1, 0.3, 0.5])
def test_p4_continuity_and_slopes(oracle, gamma):
    e = 1e-9
    assert oracle.W(gamma - e, gamma) == pytest.approx(float(oracle.W(gamma + e, gamma)), abs=1e-8)
    assert oracle.W(1.0 - e, gamma) == pytest.approx(1.0, abs=1e-8)
    h = 1e-4
    slope1 = (1.0 - oracle.W(1.0 - h, gamma)) / h          # W'(1-) = 0
    assert abs(slope1) < 1e-6
    slope_g = (oracle.W(gamma + h, gamma) - oracle.W(gamma, gamma)) / h   # W'(gamma+) = C_in
    assert slope_g == pytest.approx(oracle.Cin(gamma), rel=1e-6)
    assert oracle.W(0.5 * gamma, gamma) == pytest.approx(0.5 * gamma * oracle.Cin(gamma), rel=1e-14)


def test_p4_golden_table(oracle):
    rows = [ln.split() for ln in open(GOLD) if not ln.startswith("#")]
    assert len(rows) >= 12
    for ys, ks, ws in rows:
        y, k, w = float(ys), float(ks), float(ws)
        assert float(oracle.K((y - 0.1) / 0.9)) == pytest.approx(k, abs=1e-14)
        assert float(oracle.W(y, 0.1)) == pytest.approx(w, abs=5e-14)


@pytest.mark.parametrize("gamma", [0.1, 0.3, 0.5])
def test_p5_closed_form_equals_quadrature(oracle, gamma):
    for y in (0.02, gamma, 0.5 * (gamma + 1), 0.77, 0.95):
        pts = [p for p in (gamma,) if y < p < 1.0]
        integral, _ = quad(lambda t: K_plain((t - gamma) / (1 - gamma)) / t**2, y, 1.0,
                           points=pts or None, epsabs=1e-13, epsrel=1e-13)
        assert float(oracle.W(y, gamma)) == pytest.approx(y * (1.0 + integral), abs=1e-11)


def test_gamma_zero_limit(oracle):
    # r_in = 0 is legal (0 <= r_in < r_out): C_in -> 7/3, W(0) = 0, W(1) = 1
    assert oracle.Cin(0.0) == pytest.approx(7.0 / 3.0)
    assert float(oracle.W(0.0, 0.0)) == pytest.approx(0.0, abs=1e-15)
    assert float(oracle.W(1.0 - 1e-12, 0.0)) == pytest.approx(1.0, abs=1e-10)
