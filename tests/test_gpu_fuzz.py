"""Seeded random cases for the whole hot path against the fp64 oracle: odd sizes, every leaf/group size,
both key widths, both walk modes, clumped and degenerate geometries.

At theta = 0 the tree path is the direct sum (north_star): accelerations and potentials must match O2 to
1e-5 per particle and the neighbour lists must equal O3 outside the 1e-6 band, whatever the tree looks
like -- so a wrong leaf range, group boundary, look-back prefix or stack hand-over shows up here.
At theta > 0 the cell terms come in: error against O2 within the workload tolerances.
"""
import os

import numpy as np
import pytest

from p3t_parity_helpers import assert_same_neighbour_sets, csr_sets, rel_err

pytestmark = pytest.mark.gpu


def _geometry(rng, kind, n):
    if kind == 0:       # uniform cube
        return rng.uniform(-1.0, 1.0, (n, 3))
    if kind == 1:       # a few tight clumps of very different sizes (deep, lopsided tree)
        k = int(rng.integers(2, 6))
        centres = rng.uniform(-1.0, 1.0, (k, 3))
        scale = 10.0 ** rng.uniform(-4.0, -0.5, k)
        which = rng.integers(0, k, n)
        return centres[which] + scale[which, None] * rng.normal(size=(n, 3))
    if kind == 2:       # thin sheet (two coordinates span the box, one is nearly constant)
        p = rng.uniform(-1.0, 1.0, (n, 3))
        p[:, int(rng.integers(0, 3))] *= 1e-5
        return p
    if kind == 3:       # lattice with repeated points (equal keys, leaves above NLEAF at the deepest level)
        g = rng.integers(0, 6, (n, 3)).astype(np.float64) / 8.0
        return g
    # centrally concentrated (Plummer-like radii)
    u = rng.uniform(1e-6, 1.0 - 1e-6, n)
    r = 0.1 / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    d = rng.normal(size=(n, 3))
    return np.clip(r[:, None] * d / np.linalg.norm(d, axis=1)[:, None], -50.0, 50.0)


# P3T_FUZZ_CASES=1200 python -m pytest tests/test_gpu_fuzz.py -q -m gpu  runs a longer campaign over the same generator
CASES = list(range(int(os.environ.get("P3T_FUZZ_CASES", "24"))))


@pytest.mark.parametrize("case", CASES)
def test_random_case_matches_oracle(oracle, case):
    from paper_1506_04553_b200 import binding

    rng = np.random.default_rng(1506_04553 + case)
    n = int(rng.choice([1, 2, 17, 63, 64, 65, 129, 1000, 1025, 2047, 3000, 4097, 6000]))
    kind = case % 5
    pos = np.ascontiguousarray(_geometry(rng, kind, n).astype(np.float32))
    mass = (rng.uniform(0.2, 1.8, n) / n).astype(np.float32)
    if case % 7 == 3:
        mass[rng.integers(0, n, max(1, n // 10))] = 0.0               # massless bodies
    extent = float(np.ptp(pos, axis=0).max()) or 1.0
    eps = np.float32(10.0 ** rng.uniform(-6.0, -2.0) * extent)
    r_out = np.float32(10.0 ** rng.uniform(-2.5, -0.7) * extent)
    r_in = np.float32(r_out * rng.choice([0.0, 0.1, 0.5]))
    h = np.float32(r_out * rng.choice([1.0, 1.2, 1.5]))
    theta = [0.0, 0.0, 0.3, 0.6][case % 4]
    nleaf = int(rng.choice([1, 2, 7, 16, 32]))
    ngroup = int(rng.choice([32, 64]))
    key_bits = int(rng.choice([30, 63]))
    mode = 1 + case % 4
    curve, merge = (case // 4) % 2, [0, 1, 2, 3, 4, 32][(case // 8) % 6]     # Morton / Peano-Hilbert keys, group merge levels
    m64, q64 = mass.astype(np.float64), pos.astype(np.float64)
    a, p = oracle.direct(m64, q64, float(eps), float(r_in), float(r_out))
    ooff, olst, band = oracle.neighbours(q64, float(eps), float(h))
    cap = max(int(ooff[-1]) + 1024, 1 << 16)
    with binding.P3T(n, key_bits=key_bits, nbr_capacity=cap) as ctx:
        ctx.set_tree_params(nleaf, ngroup)
        ctx.set_walk_mode(mode)
        ctx.set_key_curve(curve)
        ctx.set_group_merge_levels(merge)
        ctx.set_params(float(eps), theta, float(r_in), float(r_out), float(h))
        ctx.soft_force(mass, pos)
        acc, pot = ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
        st = ctx.get_stats()
    info = f"case {case}: n={n} kind={kind} theta={theta} nleaf={nleaf} ngroup={ngroup} keys={key_bits} mode={mode} curve={curve} merge={merge}"
    assert_same_neighbour_sets(csr_sets(off, nbr), csr_sets(ooff, olst), band)
    assert st["n_neighbours"] == len(nbr), info
    if n == 1:
        assert np.all(acc == 0) and np.all(pot == 0), info
        return
    # scale of the comparison: the particle's own force, floored by the typical force (a particle at a
    # symmetric spot has |a| far below the sum of the magnitudes of its terms)
    an = np.linalg.norm(a, axis=1)
    floor = np.median(an)
    err = np.linalg.norm(acc.astype(np.float64) - a, axis=1) / np.maximum(an, floor)
    perr = np.abs(pot.astype(np.float64) - p) / np.maximum(np.abs(p), np.median(np.abs(p)))
    if theta == 0.0:
        assert st["n_pc"] == 0, info
        assert err.max() <= 1e-5 and perr.max() <= 1e-5, info + f" err {err.max():.2e} {perr.max():.2e}"
    else:
        # north_star: within 1e-3 / 1e-2 at the workload theta (0.4 - 0.5) "and no worse than the CPU tree oracle at the same
        # theta".  theta = 0.6 is beyond the workloads: on the lattice geometry (216 distinct points, forces that nearly cancel)
        # the METHOD's median error is 2e-3, the same for O4, so beyond the fixed bounds the second clause decides (10 % margin:
        # the two trees are different instances of the same rule -- padded cube, key-built cells -- and differ by a few per cent).
        med, p99 = 1e-3, 1e-2
        if np.median(err) > med or np.percentile(err, 99) > p99:
            o4 = oracle.Tree(m64, q64, nleaf=nleaf).walk(float(eps), theta, float(r_in), float(r_out), float(h))
            oerr = np.linalg.norm(o4["acc"] - a, axis=1) / np.maximum(an, floor)
            med, p99 = max(med, 1.1 * np.median(oerr)), max(p99, 1.1 * np.percentile(oerr, 99))
        assert np.median(err) <= med and np.percentile(err, 99) <= p99, info + f" {np.median(err):.2e} {np.percentile(err, 99):.2e}"
        assert np.median(perr) <= 1e-3 and np.percentile(perr, 99) <= 1e-2, info


@pytest.mark.parametrize("kind,n,mode", [(1, 150001, 1), (3, 70000, 2), (4, 262145, 1)])
def test_large_random_case_on_a_target_subset(oracle, kind, n, mode):
    """Many build tiles and sort tiles (look-back chains, carried cuts, ragged last tile), theta = 0, checked
    on 512 seeded targets."""
    from paper_1506_04553_b200 import binding

    rng = np.random.default_rng(7 * n + kind)
    pos = np.ascontiguousarray(_geometry(rng, kind, n).astype(np.float32))
    mass = (rng.uniform(0.2, 1.8, n) / n).astype(np.float32)
    extent = float(np.ptp(pos, axis=0).max())
    eps, r_out = np.float32(1e-6 * extent), np.float32({1: 2e-5, 3: 3e-3, 4: 1e-4}[kind] * extent)   # lists stay short
    r_in, h = np.float32(0.1 * r_out), np.float32(1.2 * r_out)
    sub = np.sort(rng.choice(n, 512, replace=False)).astype(np.int64)
    m64, q64 = mass.astype(np.float64), pos.astype(np.float64)
    a, p = oracle.direct(m64, q64, float(eps), float(r_in), float(r_out), subset=sub)
    ooff, olst, band = oracle.neighbours(q64, float(eps), float(h), subset=sub)
    with binding.P3T(n, key_bits=63, nbr_capacity=1 << 27) as ctx:
        ctx.set_walk_mode(mode)
        ctx.set_params(float(eps), 0.0, float(r_in), float(r_out), float(h))
        ctx.soft_force(mass, pos)
        acc, pot = ctx.get_acc_pot()
        off, nbr = ctx.get_neighbours()
    assert_same_neighbour_sets(csr_sets(off, nbr, sub), csr_sets(ooff, olst), band, ids=sub)
    an = np.linalg.norm(a, axis=1)
    err = np.linalg.norm(acc[sub].astype(np.float64) - a, axis=1) / np.maximum(an, np.median(an))
    perr = np.abs(pot[sub].astype(np.float64) - p) / np.abs(p)
    assert err.max() <= 1e-5 and perr.max() <= 1e-5, (err.max(), perr.max())
