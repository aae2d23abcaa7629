"""TEST INFRASTRUCTURE ONLY -- oracle for rows a2, a5 and a6 of the hot path.

Plain numpy / pure-Python restatement of
  a2  Morton keys: quantise to `max_level` bits per dimension relative to the root cube and
      interleave (x most significant)                                  -- north_star; A11
      Peano-Hilbert keys: the same quantised cell coordinates taken through the transform of J. Skilling,
      "Programming the Hilbert curve" (AIP Conf. Proc. 707, 2004: AxestoTranspose / TransposetoAxes), then
      interleaved the same way.  Both curves visit the same octree cells (a level-l cell is a run of keys
      sharing their top 3 l bits); they differ in the order of the octants inside a cell       -- DESIGN.md A25
  a5  octree from the sorted keys: a cell (a maximal run of keys sharing a 3*level-bit prefix) with
      more than NLEAF bodies is split into its non-empty octants, until <= NLEAF or level =
      max_level ("Barnes-Hut tree"; leaf capacity and depth: DESIGN.md A11)
  a6  cell moments from the body range: mass, centre of mass, traceful quadrupole about the
      centre of mass, tight AABB ("up to the quadrupole moment"; A8)
by recursion over index ranges -- no window tricks, no level-major scans, nothing shared with
paper_1506_04553_b200/csrc.  Imported only by tests/.

Pins (tests/test_oracle_keytree.py): the key-built tree has the same leaves (as body sets) as the
pointer-based octree of p3t_oracle.c built by geometric bisection of the same cube; Morton order is
the order of a depth-first octant traversal; keys of a 2x2x2 lattice are 0..7 in (x,y,z) bit order.
The quantisation is a floating-point decision of an integer: it is taken in fp32 (the kernel's
precision) from the cube the caller passes, as the parity rules require.
"""
from __future__ import annotations

import numpy as np


def root_cube(pos):
    """Root cube (A11): centre = midpoint of the position AABB, side = largest extent.
    Returns (min_corner[3], side) in fp64 WITHOUT padding; callers compare with a tolerance."""
    q = np.asarray(pos, dtype=np.float64).reshape(-1, 3)
    lo, hi = q.min(axis=0), q.max(axis=0)
    side = float((hi - lo).max())
    return 0.5 * (lo + hi) - 0.5 * side, side


def _interleave(cells, max_level):
    key = np.zeros(cells[0].shape[0], dtype=np.uint64)
    for k in range(max_level):
        for d, sh in ((0, 2), (1, 1), (2, 0)):
            bit = (cells[d] >> np.uint64(k)) & np.uint64(1)
            key |= bit << np.uint64(3 * k + sh)
    return key


def quantise(pos, cube_min, side, max_level, dtype=np.float32):
    """Integer cell coordinates (three uint64 arrays) of positions at the finest level, as morton_keys takes them."""
    ft = np.dtype(dtype).type
    q = np.asarray(pos, dtype=dtype).reshape(-1, 3)
    cmin = np.asarray(cube_min, dtype=dtype)
    scale = ft(ft(1 << max_level) / ft(side))
    qmax = (1 << max_level) - 1
    cells = []
    for d in range(3):
        t = np.maximum((q[:, d] - cmin[d]) * scale, ft(0.0))
        cells.append(np.minimum(t.astype(np.int64), qmax).astype(np.uint64))
    return cells


def hilbert_keys(pos, cube_min, side, max_level, dtype=np.float32):
    """Peano-Hilbert keys: Skilling's AxestoTranspose on the quantised coordinates, written out for arrays, then
    the bits interleaved as in morton_keys (X[0] most significant in every triple)."""
    X = quantise(pos, cube_min, side, max_level, dtype)
    one = np.uint64(1)
    M = one << np.uint64(max_level - 1)
    Q = M
    while Q > one:                                   # "inverse undo"
        P = Q - one
        for i in range(3):
            hit = (X[i] & Q) != 0
            t = np.where(hit, np.uint64(0), (X[0] ^ X[i]) & P)
            X[0] = np.where(hit, X[0] ^ P, X[0] ^ t)   # invert / exchange
            X[i] = X[i] ^ t if i else X[0]
        Q >>= one
    for i in range(1, 3):                            # Gray encode
        X[i] = X[i] ^ X[i - 1]
    t = np.zeros_like(X[0])
    Q = M
    while Q > one:
        t = np.where((X[2] & Q) != 0, t ^ (Q - one), t)
        Q >>= one
    return _interleave([x ^ t for x in X], max_level)


def hilbert_decode(key, max_level):
    """Integer cell coordinates (ix, iy, iz) of one key: Skilling's TransposetoAxes, python ints."""
    key = int(key)
    X = [0, 0, 0]
    for k in range(max_level):
        for d, sh in ((0, 2), (1, 1), (2, 0)):
            X[d] |= ((key >> (3 * k + sh)) & 1) << k
    N = 2 << (max_level - 1)
    t = X[2] >> 1                                    # Gray decode
    for i in (2, 1):
        X[i] ^= X[i - 1]
    X[0] ^= t
    Q = 2
    while Q != N:                                    # undo excess work
        P = Q - 1
        for i in (2, 1, 0):
            if X[i] & Q:
                X[0] ^= P
            else:
                t = (X[0] ^ X[i]) & P
                X[0] ^= t
                X[i] ^= t
        Q <<= 1
    return tuple(X)


def morton_keys(pos, cube_min, side, max_level, dtype=np.float32):
    """Keys of positions for the given cube; bit (3k+2, 3k+1, 3k) = bit k of (x, y, z).
    dtype = the precision the quantisation is taken in (fp32 = the kernel's; fp64 for the pins)."""
    ft = np.dtype(dtype).type
    q = np.asarray(pos, dtype=dtype).reshape(-1, 3)
    cmin = np.asarray(cube_min, dtype=dtype)
    scale = ft(ft(1 << max_level) / ft(side))
    qmax = (1 << max_level) - 1
    cells = []
    for d in range(3):
        t = (q[:, d] - cmin[d]) * scale            # one subtract, one multiply in `dtype`
        t = np.maximum(t, ft(0.0))
        c = np.minimum(t.astype(np.int64), qmax)    # truncation toward zero
        cells.append(c.astype(np.uint64))
    key = np.zeros(q.shape[0], dtype=np.uint64)
    for k in range(max_level):
        for d, sh in ((0, 2), (1, 1), (2, 0)):
            bit = (cells[d] >> np.uint64(k)) & np.uint64(1)
            key |= bit << np.uint64(3 * k + sh)
    return key


def build_cells(keys_sorted, nleaf, max_level):
    """Octree over sorted keys.  Returns a list of dicts (level, start, count, leaf, parent, children)
    numbered level by level, each level in body order (so children are contiguous)."""
    keys = [int(k) for k in keys_sorted]
    n = len(keys)
    cells = [dict(level=0, start=0, count=n, parent=-1)]
    frontier = [0]
    while frontier:
        nxt = []
        for ci in frontier:
            c = cells[ci]
            L, s, cnt = c["level"], c["start"], c["count"]
            if cnt <= nleaf or L == max_level:
                c["leaf"], c["children"] = True, []
                continue
            c["leaf"], c["children"] = False, []
            shift = 3 * (max_level - (L + 1))
            a = s
            while a < s + cnt:
                octant = keys[a] >> shift
                b = a
                while b < s + cnt and (keys[b] >> shift) == octant:
                    b += 1
                cells.append(dict(level=L + 1, start=a, count=b - a, parent=ci))
                c["children"].append(len(cells) - 1)
                nxt.append(len(cells) - 1)
                a = b
        frontier = nxt
    return cells


def cell_geometry(cell, key, cube_min, side, max_level, curve="morton"):
    """Geometric centre and side of a cell from the key of any of its bodies."""
    L = cell["level"]
    l = side / (1 << L)
    if curve == "hilbert":
        ix, iy, iz = (c >> (max_level - L) for c in hilbert_decode(key, max_level))
        g = np.asarray(cube_min, dtype=np.float64) + (np.array([ix, iy, iz]) + 0.5) * l
        return g, l
    pre = int(key) >> (3 * (max_level - L)) if L else 0
    ix = iy = iz = 0
    for k in range(L):
        iz |= ((pre >> (3 * k)) & 1) << k
        iy |= ((pre >> (3 * k + 1)) & 1) << k
        ix |= ((pre >> (3 * k + 2)) & 1) << k
    g = np.asarray(cube_min, dtype=np.float64) + (np.array([ix, iy, iz]) + 0.5) * l
    return g, l


def moments(bodies, start, count):
    """M, centre of mass c, traceful Q_ab = sum m (x-c)_a (x-c)_b (xx,yy,zz,xy,xz,yz), AABB; fp64."""
    b = np.asarray(bodies, dtype=np.float64)[start:start + count]
    m, x = b[:, 3], b[:, :3]
    M = m.sum()
    c = (m[:, None] * x).sum(axis=0) / M if M > 0 else 0.5 * (x.min(axis=0) + x.max(axis=0))
    r = x - c
    Q = np.array([(m * r[:, 0] * r[:, 0]).sum(), (m * r[:, 1] * r[:, 1]).sum(), (m * r[:, 2] * r[:, 2]).sum(),
                  (m * r[:, 0] * r[:, 1]).sum(), (m * r[:, 0] * r[:, 2]).sum(), (m * r[:, 1] * r[:, 2]).sum()])
    return M, c, Q, x.min(axis=0), x.max(axis=0)
