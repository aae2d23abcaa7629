"""Pins for oracle/keytree.py (rows a2, a5, a6): Morton keys, octree from sorted keys, moments.

The key-built tree is pinned against the independent pointer-based octree of p3t_oracle.c (built by
geometric bisection, no keys, no sort): same cube -> same leaves as body sets, same cell count.
"""
import numpy as np
import pytest

from oracle import keytree
from paper_1506_04553_b200 import workloads


def test_lattice_keys_are_octant_numbers():
    pts = np.array([[x, y, z] for x in (0.25, 0.75) for y in (0.25, 0.75) for z in (0.25, 0.75)])
    keys = keytree.morton_keys(pts, [0, 0, 0], 1.0, 1)
    assert keys.tolist() == list(range(8))                    # x is the most significant bit
    keys3 = keytree.morton_keys(pts, [0, 0, 0], 1.0, 3)
    assert (keys3 >> np.uint64(6)).tolist() == list(range(8))  # the top level is still the octant


def test_key_order_is_depth_first_octant_order():
    rng = np.random.default_rng(3)
    p = rng.uniform(0, 1, (500, 3))
    k = keytree.morton_keys(p, [0, 0, 0], 1.0, 10, dtype=np.float64)
    # brute force: compare two points by the first level on which their octants differ
    def octants(q):
        out = []
        lo = np.zeros(3); side = 1.0
        for _ in range(10):
            side /= 2
            o = 0
            for d in range(3):
                bit = int(q[d] >= lo[d] + side)
                lo[d] += bit * side
                o = (o << 1) | bit
            out.append(o)
        return out
    order = np.argsort(k, kind="stable")
    paths = [octants(p[i]) for i in order]
    assert paths == sorted(paths)


@pytest.mark.parametrize("b", [1, 2, 3, 4])
def test_hilbert_keys_visit_a_lattice_once_and_move_to_a_face_neighbour_each_step(b):
    """What makes a curve a Hilbert curve: a bijection of the 8^b cells onto 0 .. 8^b - 1 whose consecutive cells share
    a face.  (Morton order fails the second half at every octant boundary.)"""
    n = 1 << b
    ijk = np.array([[x, y, z] for x in range(n) for y in range(n) for z in range(n)])
    pts = (ijk + 0.5) / n
    k = keytree.hilbert_keys(pts, [0, 0, 0], 1.0, b, dtype=np.float64)
    assert sorted(k.tolist()) == list(range(8 ** b))
    path = ijk[np.argsort(k)]
    assert np.all(np.abs(np.diff(path, axis=0)).sum(axis=1) == 1)
    assert path[0].tolist() == [0, 0, 0]
    km = keytree.morton_keys(pts, [0, 0, 0], 1.0, b, dtype=np.float64)
    if b > 1:
        assert np.any(np.abs(np.diff(ijk[np.argsort(km)], axis=0)).sum(axis=1) > 1)
    for key, c in zip(k, ijk):                                   # the inverse transform gives the cell back
        assert keytree.hilbert_decode(key, b) == tuple(c)


def test_hilbert_and_morton_keys_have_the_same_cells_at_every_level():
    """A level-l cell is the set of bodies with equal top 3 l key bits, for both curves: the octree built from either
    key is the same tree (only the order of the children differs)."""
    rng = np.random.default_rng(9)
    p = rng.uniform(0, 1, (4000, 3)) ** 2                       # clustered towards a corner: deep levels get used
    L = 21
    kh = keytree.hilbert_keys(p, [0, 0, 0], 1.0, L, dtype=np.float64)
    km = keytree.morton_keys(p, [0, 0, 0], 1.0, L, dtype=np.float64)
    cells = keytree.quantise(p, [0, 0, 0], 1.0, L, dtype=np.float64)
    for l in (1, 2, 5, 9, 14, 21):
        sh = np.uint64(3 * (L - l))
        pairs = set(zip((kh >> sh).tolist(), (km >> sh).tolist()))
        assert len(pairs) == len({a for a, _ in pairs}) == len({b for _, b in pairs})
    for i in range(0, 4000, 97):
        assert keytree.hilbert_decode(kh[i], L) == tuple(int(c[i]) for c in cells)
    # 10-bit keys are the top 30 bits' worth of the same construction on the coarser lattice
    k10 = keytree.hilbert_keys(p, [0, 0, 0], 1.0, 10, dtype=np.float64)
    assert np.array_equal(k10, kh >> np.uint64(33))


@pytest.mark.parametrize("curve", ["morton", "hilbert"])
@pytest.mark.parametrize("nleaf,max_level", [(16, 10), (4, 21), (1, 21)])
def test_key_tree_equals_pointer_tree(oracle, nleaf, max_level, curve):
    c = workloads.config(1, n=3000)
    m, q = c["mass"].astype(np.float64), c["pos"].astype(np.float64)
    t = oracle.Tree(m, q, nleaf=nleaf, max_depth=max_level)
    nd = t.nodes()
    side = nd["side"][0]
    cmin = nd["g"][0] - 0.5 * side
    keys = (keytree.hilbert_keys if curve == "hilbert" else keytree.morton_keys)(q, cmin, side, max_level, dtype=np.float64)
    order = np.argsort(keys, kind="stable")
    cells = keytree.build_cells(keys[order], nleaf, max_level)
    assert len(cells) == t.nnodes
    perm = t.perm()
    leaves_ptr = {frozenset(perm[f:f + n].tolist()) for f, n, lf in zip(nd["first"], nd["count"], nd["leaf"]) if lf}
    leaves_key = {frozenset(order[x["start"]:x["start"] + x["count"]].tolist()) for x in cells if x["leaf"]}
    assert leaves_ptr == leaves_key
    # geometry from the key prefix equals the bisection geometry
    geo_ptr = {(int(l), tuple(np.round(g / side, 9))) for l, g in zip(nd["level"], nd["g"])}
    geo_key = set()
    for x in cells:
        g, l = keytree.cell_geometry(x, keys[order][x["start"]], cmin, side, max_level, curve=curve)
        geo_key.add((x["level"], tuple(np.round(g / side, 9))))
    assert geo_ptr == geo_key


def test_cells_partition_and_numbering():
    rng = np.random.default_rng(5)
    keys = np.sort(rng.integers(0, 1 << 30, 2000, dtype=np.uint64))
    keys[100:140] = keys[100]                                  # coincident keys: a max-depth leaf > nleaf
    keys = np.sort(keys)
    cells = keytree.build_cells(keys, 8, 10)
    covered = np.zeros(2000, dtype=int)
    for i, c in enumerate(cells):
        if c["leaf"]:
            covered[c["start"]:c["start"] + c["count"]] += 1
            assert c["count"] <= 8 or c["level"] == 10
        else:
            ch = c["children"]
            assert ch == list(range(ch[0], ch[0] + len(ch)))   # contiguous
            assert sum(cells[k]["count"] for k in ch) == c["count"]
            assert cells[ch[0]]["start"] == c["start"]
            assert all(cells[k]["level"] == c["level"] + 1 and cells[k]["parent"] == i for k in ch)
    assert np.all(covered == 1)
    assert max(c["count"] for c in cells if c["leaf"]) >= 40
    levels = [c["level"] for c in cells]
    assert levels == sorted(levels)


def test_moments_match_pointer_tree(oracle):
    c = workloads.config(3, n=2000)
    m, q = c["mass"].astype(np.float64), c["pos"].astype(np.float64)
    t = oracle.Tree(m, q, nleaf=16, max_depth=21)
    nd = t.nodes()
    perm = t.perm()
    bodies = np.concatenate([q[perm], m[perm, None]], axis=1)
    for k in range(0, t.nnodes, 7):
        M, com, Q, lo, hi = keytree.moments(bodies, int(nd["first"][k]), int(nd["count"][k]))
        np.testing.assert_allclose(M, nd["M"][k], rtol=1e-13)
        np.testing.assert_allclose(com, nd["c"][k], rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(Q, nd["Q"][k], rtol=1e-9, atol=1e-18)
        np.testing.assert_allclose(lo, nd["bmin"][k]); np.testing.assert_allclose(hi, nd["bmax"][k])
