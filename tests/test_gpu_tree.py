"""GPU parity for rows a1-a6 (bounding cube, Morton keys, radix sort, gather, octree, moments).

Integer / index work is compared bit-exactly with oracle/keytree.py; moments within fp32 tolerances
of the fp64 recomputation from the body ranges.  Everything goes through the C ABI.
"""
import numpy as np
import pytest

from paper_1506_04553_b200 import workloads

pytestmark = pytest.mark.gpu

LEAF = 0x80000000


def _build(cfg, key_bits=None, nleaf=16, ngroup=64, theta=None, curve="hilbert"):
    from paper_1506_04553_b200 import binding

    kb = key_bits or cfg["key_bits"]
    ctx = binding.P3T(cfg["n"], key_bits=kb)
    ctx.set_key_curve(curve)
    ctx.set_params(cfg["eps"], cfg["theta"] if theta is None else theta, cfg["r_in"], cfg["r_out"], cfg["r_search"])
    ctx.set_tree_params(nleaf, ngroup)
    ctx.load_particles(cfg["mass"], cfg["pos"])
    ctx.build_tree()
    ctx.synchronize()
    return ctx, (21 if kb == 63 else 10)


CASES = [  # (config, n, key_bits, nleaf, ngroup)
    (1, 4096, 30, 16, 64), (1, 4096, 63, 16, 32), (1, 5000, 63, 8, 64), (3, 20011, 63, 16, 64),
    (4, 30000, 63, 16, 64), (1, 100, 30, 1, 32), (1, 7, 63, 16, 64),
]


@pytest.mark.parametrize("curve", ["morton", "hilbert"])
@pytest.mark.parametrize("k,n,kb,nleaf,ngroup", CASES)
def test_keys_sort_octree_match_keytree_oracle(k, n, kb, nleaf, ngroup, curve):
    from oracle import keytree

    cfg = workloads.config(k, n=n)
    ctx, max_level = _build(cfg, kb, nleaf, ngroup, curve=curve)
    cube = ctx.array("root_cube")
    # a1: the cube is the oracle's definition (centre = AABB midpoint, side = largest extent), padded
    cmin, side = keytree.root_cube(cfg["pos"])
    assert side <= cube[3] <= side * (1 + 1e-5)
    np.testing.assert_allclose(cube[:3] + 0.5 * cube[3], cmin + 0.5 * side, atol=2e-6 * side)
    assert np.all(cfg["pos"] >= cube[:3]) and np.all(cfg["pos"] < cube[:3] + cube[3])
    # a2-a3: keys bit-exact, sorted; a4: permutation and gathered bodies
    keys = ctx.array("keys")
    idx = ctx.array("sorted_idx")
    ref = (keytree.hilbert_keys if curve == "hilbert" else keytree.morton_keys)(cfg["pos"], cube[:3], cube[3], max_level)
    assert np.array_equal(np.sort(idx), np.arange(n, dtype=np.uint32))
    assert np.array_equal(keys, ref[idx])
    assert np.all(keys[1:] >= keys[:-1])
    order = np.argsort(ref, kind="stable")                     # LSD radix sort is stable
    assert np.array_equal(idx, order.astype(np.uint32))
    bodies = ctx.array("bodies")
    assert np.array_equal(bodies[:, :3], cfg["pos"][idx]) and np.array_equal(bodies[:, 3], cfg["mass"][idx])
    # a5: cells identical to the recursive construction, in the same numbering
    cells = keytree.build_cells(keys, nleaf, max_level)
    st = ctx.get_stats()
    assert st["n_cells"] == len(cells)
    assert st["n_leaves"] == sum(c["leaf"] for c in cells)
    assert st["depth"] == max(c["level"] for c in cells)
    level, start, parent, meta = ctx.array("cell_level"), ctx.array("cell_start"), ctx.array("cell_parent"), ctx.array("cell_meta")
    assert np.array_equal(level, np.array([c["level"] for c in cells], dtype=np.uint8))
    assert np.array_equal(start, np.array([c["start"] for c in cells], dtype=np.uint32))
    assert np.array_equal(parent.astype(np.int64), np.array([c["parent"] if c["parent"] >= 0 else 0xffffffff for c in cells]))
    for i, c in enumerate(cells):
        if c["leaf"]:
            assert meta[i, 0] == c["start"] and meta[i, 1] == (c["count"] | LEAF)
        else:
            assert meta[i, 0] == c["children"][0] and meta[i, 1] == len(c["children"])
    # groups: a partition of the sorted bodies into runs of <= ngroup
    gs = ctx.array("group_start").astype(np.int64)
    assert st["n_groups"] == len(gs) - 1
    assert gs[0] == 0 and gs[-1] == n and np.all(np.diff(gs) >= 1) and np.all(np.diff(gs) <= ngroup)
    ctx.close()


@pytest.mark.parametrize("curve", ["morton", "hilbert"])
@pytest.mark.parametrize("k,n,kb", [(1, 4096, 30), (3, 20011, 63), (4, 30000, 63)])
def test_moments_match_fp64_recomputation(k, n, kb, curve):
    from oracle import keytree

    cfg = workloads.config(k, n=n)
    ctx, max_level = _build(cfg, kb, curve=curve)
    keys, bodies, cube = ctx.array("keys"), ctx.array("bodies"), ctx.array("root_cube")
    cells = keytree.build_cells(keys, 16, max_level)
    mac, m0, m1 = ctx.array("cell_mac"), ctx.array("cell_mom0"), ctx.array("cell_mom1")
    bmin, bmax = ctx.array("cell_bmin"), ctx.array("cell_bmax")
    theta, h = cfg["theta"], cfg["r_search"]
    rng = np.random.default_rng(1)
    pick = np.unique(np.concatenate([np.arange(min(64, len(cells))), rng.integers(0, len(cells), 1500)]))
    for i in pick:
        c = cells[i]
        M, com, Q, lo, hi = keytree.moments(bodies, c["start"], c["count"])
        ext = max(float((hi - lo).max()), 1e-30)
        assert abs(m0[i, 0] - M) <= 2e-6 * M
        np.testing.assert_allclose(mac[i, :3], com, atol=3e-6 * ext + 2e-7 * np.abs(com).max())
        qscale = M * ext * ext
        np.testing.assert_allclose(np.concatenate([m0[i, 1:], m1[i, :3]]), Q, atol=2e-5 * qscale + 1e-30)
        assert np.array_equal(bmin[i, :3], lo.astype(np.float32)) and np.array_equal(bmax[i, :3], hi.astype(np.float32))
        # acceptance radius: never below either clause of R-MAC (A9, A10)
        g, l = keytree.cell_geometry(c, keys[c["start"]], cube[:3], cube[3], max_level, curve=curve)
        delta = np.linalg.norm(com - g)
        rmax = np.linalg.norm(bodies[c["start"]:c["start"] + c["count"], :3].astype(np.float64) - com, axis=1).max()
        rc = np.sqrt(float(mac[i, 3]))
        assert rc >= (l / theta + delta) * (1 - 1e-5)
        assert rc >= h + rmax
        assert rc <= max(l / theta + delta, h + 1.7321 * ext + 1e-30) * (1 + 1e-3) + 1e-4 * cube[3]
    # root: total mass and centre of mass of everything
    np.testing.assert_allclose(m0[0, 0], cfg["mass"].astype(np.float64).sum(), rtol=2e-6)
    ctx.close()


def test_coincident_points_make_a_deep_leaf():
    from oracle import keytree

    cfg = workloads.config(1, n=2000)
    cfg["pos"][100:160] = cfg["pos"][100]                       # 60 bodies at one point
    ctx, max_level = _build(cfg, 63)
    keys = ctx.array("keys")
    cells = keytree.build_cells(keys, 16, max_level)
    meta, level = ctx.array("cell_meta"), ctx.array("cell_level")
    assert ctx.get_stats()["n_cells"] == len(cells)
    big = [(int(meta[i, 1]) & 0x7fffffff, int(level[i])) for i in range(len(cells)) if int(meta[i, 1]) & LEAF and (int(meta[i, 1]) & 0x7fffffff) > 16]
    assert big == [(60, 21)]
    ctx.close()


def test_rebuilding_one_tree_300_times_gives_the_same_bits():
    """Repeat-stress of the inter-CTA protocols racecheck cannot see (global memory): the radix sort's relaxed look-back
    words, the build's look-back columns and the moments climb (release fence + relaxed arrival counter, children read
    back from L2).  One 200K-body tree is rebuilt 300 times; sorted order, cell topology, groups AND moments must be
    bitwise identical every time (PAPER.md L142-153 is the GPU procedure these kernels implement)."""
    cfg = workloads.config(3, n=200003)
    ctx, _ = _build(cfg, 63)
    names = ["root_cube", "keys", "sorted_idx", "bodies", "cell_meta", "cell_level", "cell_start", "cell_parent", "group_start",
             "cell_mac", "cell_mom0", "cell_mom1", "cell_bmin", "cell_bmax"]
    first = {k: ctx.array(k).copy() for k in names}
    st0 = ctx.get_stats()
    assert st0["n_cells"] > 20000 and st0["depth"] >= 8
    for it in range(300):
        if it % 3 == 0:
            ctx.load_particles(cfg["mass"], cfg["pos"])         # also re-runs pack + bounding cube
        else:
            ctx.set_params(cfg["eps"], cfg["theta"], cfg["r_in"], cfg["r_out"], cfg["r_search"])   # invalidates the tree
        ctx.build_tree()
        st = ctx.get_stats()
        assert (st["n_cells"], st["n_leaves"], st["n_groups"], st["depth"]) == (st0["n_cells"], st0["n_leaves"], st0["n_groups"], st0["depth"])
        for k in names:
            got = ctx.array(k)
            assert got.tobytes() == first[k].tobytes(), f"rebuild {it}: {k} differs"
    ctx.close()


def _sorted_order_case(kind, n, rng):
    """Positions that make runs of keys equal on the upper bits short, long or huge."""
    if kind == "plummer":
        return workloads.config(3, n=n)["pos"]
    if kind == "clump":          # most bodies in a ball of 1e-4 of the cube: they share the upper 13 levels
        p = rng.normal(size=(n, 3)) * 1e-4
        p[:8] = rng.uniform(-1, 1, (8, 3))
        return p.astype(np.float32)
    if kind == "coincident":     # three points hold nearly everybody: runs of equal FULL keys, a third of n long
        p = np.repeat(rng.uniform(-1, 1, (3, 3)), (n + 2) // 3, axis=0)[:n]
        p[:50] = rng.uniform(-1, 1, (50, 3))
        return p[rng.permutation(n)].astype(np.float32)
    if kind == "lattice":        # repeated points: equal full keys (order by index) next to distinct ones
        return (rng.integers(0, 12, (n, 3)) / 16.0 + rng.integers(0, 2, (n, 1)) * rng.uniform(0, 1e-6, (n, 3))).astype(np.float32)
    raise ValueError(kind)


@pytest.mark.parametrize("kind,n,kb,passes", [
    ("plummer", 50000, 63, 0), ("plummer", 50000, 63, 5), ("plummer", 50000, 63, 3), ("plummer", 200003, 63, 4),
    ("clump", 30000, 63, 0), ("clump", 30000, 63, 4), ("clump", 300000, 63, 2), ("clump", 5000, 63, 1),
    ("lattice", 40000, 63, 0), ("lattice", 40000, 63, 2), ("lattice", 3000, 30, 2), ("plummer", 20000, 30, 3),
    ("plummer", 1, 63, 1), ("plummer", 33, 63, 1), ("clump", 4097, 63, 1), ("coincident", 400000, 63, 0), ("coincident", 9000, 63, 8),
])
@pytest.mark.parametrize("curve", ["morton", "hilbert"])
def test_radix_passes_over_the_upper_digits_give_the_full_stable_order(kind, n, kb, passes, curve):
    """p3t_set_sort_passes: whatever the number of radix passes, the build ends with the stable order of the FULL keys
    (runs of keys equal on the sorted bits: one thread up to 32 keys, one CTA in shared memory up to 2048, one CTA in
    global memory beyond), and a second build on the same context -- whose plan has seen the first one's runs -- too."""
    from oracle import keytree
    from paper_1506_04553_b200 import binding

    rng = np.random.default_rng(n + passes)
    pos = np.ascontiguousarray(_sorted_order_case(kind, n, rng))
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    max_level = 21 if kb == 63 else 10
    with binding.P3T(n, key_bits=kb) as ctx:
        ctx.set_key_curve(curve)
        ctx.set_sort_passes(passes)
        ctx.set_params(1e-6, 0.4, 1e-4, 1e-3, 1.2e-3)
        used = []
        for rebuild in range(3):
            ctx.load_particles(mass, pos)
            ctx.build_tree()
            ctx.synchronize()
            cube = ctx.array("root_cube")
            ref = (keytree.hilbert_keys if curve == "hilbert" else keytree.morton_keys)(pos, cube[:3], cube[3], max_level)
            idx, keys = ctx.array("sorted_idx"), ctx.array("keys")
            assert np.array_equal(idx, np.argsort(ref, kind="stable").astype(np.uint32)), (kind, n, passes, rebuild)
            assert np.array_equal(keys, ref[idx])
            st = ctx.get_stats()
            used.append((st["sort_passes"], st["sort_max_run"]))
            bodies = ctx.array("bodies")
            assert np.array_equal(bodies[:, :3], pos[idx])
        total = 8 if kb == 63 else 4
        if passes:
            assert all(u[0] == min(passes, total) for u in used), used
        elif kb == 30:
            assert all(u[0] == 4 for u in used), used
        else:
            assert all(1 <= u[0] <= 8 for u in used) and used[0][0] <= used[1][0] <= used[2][0], used   # the plan only grows
            if kind == "clump":
                assert used[0][1] > 24 and used[1][0] > used[0][0], used      # long runs seen: more passes next time
