"""Seeded synthetic workloads (the five BASELINE.json configs).

This module only generates INPUT DATA (masses, positions, velocities, the
parameter set of each config).  It holds none of the method's arithmetic and
is the one module shared by the CUDA path's callers (tests, bench.py) and the
oracle's callers.  numpy only; no torch, no CUDA.

Paper context: every workload of arXiv 1506.04553 is a generated Plummer
model in N-body units (M = 1, G = 1, E = -1/4); nothing
stands in for a dataset.  The King W0=9 model (config 4) and the Salpeter
mass function (config 3) come from BASELINE.json, not from the paper.
Recipe: DESIGN.md section 5.
"""
from __future__ import annotations

import math

import numpy as np

SEED_BASE = 150604553            # + config number
PLUMMER_A = 3.0 * math.pi / 16.0  # scale length giving E = -1/4 for M = G = 1
SIGMA_3D = 1.0 / math.sqrt(2.0)   # global 3-D velocity dispersion


def _isotropic(rng, n):
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * math.pi, n)
    s = np.sqrt(1.0 - z * z)
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def plummer(n, seed, rmax_over_a=20.0):
    """Plummer sphere positions/velocities (fp64), equal weights.

    Radius by inverting M(<r)/M = (r/a)^3 (1 + (r/a)^2)^(-3/2); bodies beyond
    rmax_over_a * a are redrawn (0.37 % of the mass); speed by rejection on
    g(q) = q^2 (1 - q^2)^(7/2), v = q * v_esc(r).  No virial rescale.
    """
    rng = np.random.default_rng(seed)
    r = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        u = rng.uniform(0.0, 1.0, todo.size)
        u = np.clip(u, 1e-300, 1.0 - 1e-16)
        rr = PLUMMER_A / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
        ok = rr <= rmax_over_a * PLUMMER_A
        r[todo[ok]] = rr[ok]
        todo = todo[~ok]
    pos = r[:, None] * _isotropic(rng, n)
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        x = rng.uniform(0.0, 1.0, todo.size)
        y = rng.uniform(0.0, 0.1, todo.size)  # max of g is 0.0923
        ok = y < x * x * (1.0 - x * x) ** 3.5
        q[todo[ok]] = x[ok]
        todo = todo[~ok]
    vesc = np.sqrt(2.0) * (r * r + PLUMMER_A ** 2) ** -0.25
    vel = (q * vesc)[:, None] * _isotropic(rng, n)
    return pos, vel


def salpeter_masses(n, seed, m_lo=0.1, m_hi=100.0, alpha=2.35):
    """dN/dm ~ m^-alpha on [m_lo, m_hi], rescaled to total mass 1."""
    rng = np.random.default_rng(seed)
    p = 1.0 - alpha
    u = rng.uniform(0.0, 1.0, n)
    m = (m_lo ** p + u * (m_hi ** p - m_lo ** p)) ** (1.0 / p)
    return m / m.sum()


def _king_profile(w0, dr=1e-3):
    """Integrate W'' + 2 W'/r = -9 rho(W)/rho(W0) outward (RK4) until W = 0."""
    from math import erf, exp, pi, sqrt

    def rho(w):
        if w <= 0.0:
            return 0.0
        return exp(w) * erf(sqrt(w)) - sqrt(4.0 * w / pi) * (1.0 + 2.0 * w / 3.0)

    rho0 = rho(w0)

    def f(r, w, dw):
        return dw, -9.0 * rho(w) / rho0 - 2.0 * dw / r

    # series start: W ~ W0 - 1.5 r^2
    r, w, dw = dr, w0 - 1.5 * dr * dr, -3.0 * dr
    rs, ws, dws = [0.0, r], [w0, w], [0.0, dw]
    while w > 0.0 and r < 1e5:
        h = dr * max(1.0, r)  # geometric step growth in the halo
        k1 = f(r, w, dw)
        k2 = f(r + h / 2, w + h / 2 * k1[0], dw + h / 2 * k1[1])
        k3 = f(r + h / 2, w + h / 2 * k2[0], dw + h / 2 * k2[1])
        k4 = f(r + h, w + h * k3[0], dw + h * k3[1])
        wn = w + h / 6 * (k1[0] + 2 * k2[0] + 2 * k3[0] + k4[0])
        dwn = dw + h / 6 * (k1[1] + 2 * k2[1] + 2 * k3[1] + k4[1])
        if wn <= 0.0:  # linear interpolation to the tidal radius
            t = w / (w - wn)
            r, dw, w = r + t * h, dw + t * (dwn - dw), 0.0
            rs.append(r); ws.append(0.0); dws.append(dw)
            break
        r, w, dw = r + h, wn, dwn
        rs.append(r); ws.append(w); dws.append(dw)
    rs, ws, dws = np.array(rs), np.array(ws), np.array(dws)
    mass = -rs * rs * dws  # G M(r) / (sigma^2 r0)
    return rs, ws, mass


def king(n, w0, seed):
    """King (1966) model, equal weights, scaled to M = 1 and U = -1/2 (G = 1)."""
    rng = np.random.default_rng(seed)
    rs, ws, mass = _king_profile(w0)
    mu = mass[-1]
    mfrac = mass / mu
    # potential energy in model units (M = 1, lengths in r0): U = -int M dM / r
    dm = np.diff(mfrac)
    rmid = 0.5 * (rs[1:] + rs[:-1])
    mmid = 0.5 * (mfrac[1:] + mfrac[:-1])
    u_model = -np.sum(mmid * dm / rmid)
    lam = 2.0 * abs(u_model)          # new length of one r0
    sigma2 = 1.0 / (lam * mu)         # from G M = -sigma^2 r0 x^2 dW/dx at the edge
    u = rng.uniform(0.0, 1.0, n)
    keep = np.concatenate([[True], np.diff(mfrac) > 0])
    x = np.interp(u, mfrac[keep], rs[keep])
    wx = np.interp(x, rs, ws)
    pos = (x * lam)[:, None] * _isotropic(rng, n)
    # speeds: f(v) ~ (exp(W - v^2/2) - 1) v^2 on v^2 < 2W, in units of sigma
    v = np.zeros(n)
    todo = np.arange(n)
    while todo.size:
        wt = wx[todo]
        vmax = np.sqrt(2.0 * wt)
        vt = rng.uniform(0.0, 1.0, todo.size) * vmax
        fmax = np.maximum(np.expm1(wt) * 2.0, 1e-300)   # bound: (e^W - 1) * v^2 e^{-v^2/2} <= (e^W - 1) * 2/e
        fv = (np.exp(wt - 0.5 * vt * vt) - 1.0) * vt * vt
        ok = rng.uniform(0.0, 1.0, todo.size) * fmax < fv
        ok |= wt <= 0.0
        v[todo[ok]] = vt[ok]
        todo = todo[~ok]
    vel = (v * math.sqrt(sigma2))[:, None] * _isotropic(rng, n)
    return pos, vel, dict(r0=lam, rt=rs[-1] * lam, sigma2=sigma2, mu=mu)


def _recentre(mass, pos, vel):
    w = mass / mass.sum()
    pos = pos - (w[:, None] * pos).sum(axis=0)
    vel = vel - (w[:, None] * vel).sum(axis=0)
    return pos, vel


def dr_buff(dt_soft):
    """Buffer shell width 3 sigma dt_soft (Table 1)."""
    return 3.0 * SIGMA_3D * dt_soft


def config(k, n=None, seed_offset=0):
    """Workload k = 1..5 of BASELINE.json (6: the SMBH-binary workload of PAPER.md L287, for the pair-class row).
    n overrides the particle count
    (used by tests to run a config's recipe at a size the oracle can afford).

    Returns a dict: mass, pos, vel as fp32 arrays (the GPU input; the oracle gets
    the same values widened to fp64) and eps, theta, r_in, r_out, r_search,
    nleaf, ngroup, key_bits, plus name / dt_soft where the config has one.
    Missing values follow DESIGN.md section 3 (readings A17).  seed_offset draws another
    realisation of the same recipe (multi.py: one independent cluster per rank).
    """
    seed = SEED_BASE + k + seed_offset
    if k == 1:
        n = n or 4096
        pos, vel = plummer(n, seed)
        mass = np.full(n, 1.0 / n)
        prm = dict(eps=1.0 / n, theta=0.5, r_out=0.01, r_search=0.012, key_bits=30, name="plummer-4k")
    elif k == 2:
        n = n or 65536
        pos, vel = plummer(n, seed)
        mass = np.full(n, 1.0 / n)
        r_out = 4.0 * n ** (-1.0 / 3.0) * 0.05
        dt = 1.0 / 256.0
        prm = dict(eps=1.0 / n, theta=0.4, r_out=r_out, r_search=r_out + dr_buff(dt), dt_soft=dt,
                   key_bits=63, name="plummer-64k-leapfrog")
    elif k == 3:
        n = n or 1048576
        pos, vel = plummer(n, seed)
        mass = salpeter_masses(n, seed + 1000)
        prm = dict(eps=1e-7, theta=0.4, r_out=0.002, r_search=0.0026, key_bits=63, name="plummer-1m-salpeter")
    elif k == 4:
        n = n or 262144
        pos, vel, _ = king(n, 9.0, seed)
        mass = np.full(n, 1.0 / n)
        prm = dict(eps=1e-7, theta=0.4, r_out=0.001, r_search=0.0013, key_bits=63, name="king-w9-256k")
    elif k == 5:
        n = n or 4194304
        pos, vel = plummer(n, seed)
        mass = np.full(n, 1.0 / n)
        prm = dict(eps=1e-7, theta=0.5, r_out=0.0015, r_search=0.00195, key_bits=63, name="plummer-4m")
    elif k == 6:
        # the SMBH-binary workload of section 3.2.2.1, not one of BASELINE.json's five: a Plummer model
        # of n field stars (mass 1 in all) plus two black holes of mass 0.01 at (+-0.5, 0, 0) with velocities
        # (0, +-0.5, 0); r_cut = 1/256 between field stars, 1/32 between a black hole and a field star, black hole
        # pairs not split; eps = 1e-4 (0 between the black holes); dt_soft = 1/1024, dr_buff = 3 sigma dt_soft
        nfs = n or 16384
        pos, vel = plummer(nfs, seed)
        mass = np.full(nfs, 1.0 / nfs)
        pos, vel = _recentre(mass, pos, vel)
        pos = np.concatenate([pos, [[0.5, 0.0, 0.0], [-0.5, 0.0, 0.0]]])
        vel = np.concatenate([vel, [[0.0, 0.5, 0.0], [0.0, -0.5, 0.0]]])
        mass = np.concatenate([mass, [0.01, 0.01]])
        n = nfs + 2
        dt = 1.0 / 1024.0
        prm = dict(eps=1e-4, theta=0.4, r_out=1.0 / 256.0, r_search=1.0 / 256.0 + dr_buff(dt), dt_soft=dt, key_bits=63,
                   name="plummer-16k-smbh-binary", classes=np.concatenate([np.zeros(nfs, np.uint8), np.ones(2, np.uint8)]),
                   class_params=dict(r_in_bf=0.1 / 32.0, r_out_bf=1.0 / 32.0, r_search_bf=1.0 / 32.0 + dr_buff(dt), eps_bb=0.0))
    else:
        raise ValueError("config must be 1..6")
    if k != 6:
        pos, vel = _recentre(mass, pos, vel)
    prm["r_in"] = 0.1 * prm["r_out"]      # gamma = 0.1 in all runs (Table 1)
    # i-groups of 32 below 40K particles (more, lighter groups fill the GPU better), 64 above (two bodies per lane: the
    # packed path; the walk splits a group over 2 or 4 warps where there are fewer groups than warps)
    prm.update(nleaf=16, ngroup=32 if n < 40000 else 64, n=n, config=k)
    # fp32 parameters: what the C ABI receives; the oracle gets these same values
    for key in ("eps", "theta", "r_in", "r_out", "r_search"):
        prm[key] = float(np.float32(prm[key]))
    if "class_params" in prm:
        prm["class_params"] = {key: float(np.float32(v)) for key, v in prm["class_params"].items()}
    prm["mass"] = mass.astype(np.float32)
    prm["pos"] = np.ascontiguousarray(pos.astype(np.float32))
    prm["vel"] = np.ascontiguousarray(vel.astype(np.float32))
    return prm
