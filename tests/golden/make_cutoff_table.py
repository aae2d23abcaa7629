"""Writes tests/golden/cutoff_gamma0p1.txt.

Independent of oracle/ AND of the paper's closed forms Eq. 16-17: W is obtained
from what Eq. 9, Eq. 12 (L85) and the end condition W(y>=1)=1
(Eq. 16 third branch, L102) fix on their own,

    K = W - y dW/dy  =>  d(W/y)/dy = -K/y^2  =>  W(y) = y [ 1 + int_y^1 K(x(t))/t^2 dt ],

by 40-digit quadrature (mpmath).  The oracle's closed-form W (Eq. 16-17 with
reading A1) must reproduce these numbers; the extracted Eq. 17 with the
denominator (1-gamma)^7 does not.

Run:  python tests/golden/make_cutoff_table.py
"""
import os

import mpmath as mp

mp.mp.dps = 40
GAMMA = mp.mpf("0.1")


def K(x):
    if x < 0:
        return mp.mpf(0)
    if x >= 1:
        return mp.mpf(1)
    return -20 * x**7 + 70 * x**6 - 84 * x**5 + 35 * x**4


def W_quadrature(y, g):
    y = mp.mpf(y)
    if y >= 1:
        return mp.mpf(1)
    pts = sorted({y, max(y, g), mp.mpf(1)})
    integral = mp.quad(lambda t: K((t - g) / (1 - g)) / t**2, pts)
    return y * (1 + integral)


def main():
    ys = ["0.05", "0.1", "0.2", "0.3", "0.4", "0.5", "0.55", "0.6", "0.7", "0.8", "0.9", "1.0", "1.5"]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cutoff_gamma0p1.txt")
    with open(out, "w") as f:
        f.write("# gamma = 0.1 (PAPER.md L100: 'for all calculations, we use gamma = 0.1')\n")
        f.write("# columns: y  K(x(y)) [Eq. 12, L85]  W(y) [Eq. 9 + Eq. 12 + W(1)=1 by quadrature]\n")
        f.write("# written by tests/golden/make_cutoff_table.py (mpmath, 40 digits)\n")
        for ys_ in ys:
            y = mp.mpf(ys_)
            k = K((y - GAMMA) / (1 - GAMMA))
            w = W_quadrature(y, GAMMA)
            f.write(f"{ys_} {mp.nstr(k, 20)} {mp.nstr(w, 20)}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
