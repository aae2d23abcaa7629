"""ctypes front end of the fp64 CPU oracle (oracle/p3t_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  The product path
(paper_1506_04553_b200) never imports this module.

All arrays are fp64; callers pass the fp32-rounded inputs widened to double so
that only arithmetic rounding separates the oracle from the GPU.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "p3t_oracle.c")
_LIB = os.path.join(_HERE, "libp3t_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, strict IEEE: no -ffast-math).

    P3T_ORACLE_SANITIZE=1 in the environment builds libp3t_oracle_san.so with AddressSanitizer and
    UndefinedBehaviorSanitizer instead (run python with LD_PRELOAD=$(gcc -print-file-name=libasan.so);
    profiles/sanitizer_r2.md has the command and its result)."""
    global _LIB
    san = os.environ.get("P3T_ORACLE_SANITIZE") == "1"
    if san:
        _LIB = os.path.join(_HERE, "libp3t_oracle_san.so")
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                 "-fno-omit-frame-pointer"] if san else ["-O2"]
        cmd = ["gcc"] + flags + ["-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _p(a, t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        d, i64, vp, i32 = C.c_double, C.c_int64, C.c_void_p, C.c_int
        pd, pi64, pi32 = C.POINTER(d), C.POINTER(i64), C.POINTER(C.c_int32)
        L.p3t_oracle_K.restype = d; L.p3t_oracle_K.argtypes = [d]
        L.p3t_oracle_Cin.restype = d; L.p3t_oracle_Cin.argtypes = [d]
        L.p3t_oracle_G.restype = d; L.p3t_oracle_G.argtypes = [d, d]
        L.p3t_oracle_W.restype = d; L.p3t_oracle_W.argtypes = [d, d]
        L.p3t_oracle_pair_weights.restype = None
        L.p3t_oracle_pair_weights.argtypes = [d, d, d, pd, pd]
        L.p3t_oracle_direct.restype = None
        L.p3t_oracle_direct.argtypes = [i64, pd, pd, d, d, d, i64, pi64, pd, pd, pd, pd]
        L.p3t_oracle_neighbours.restype = i64
        L.p3t_oracle_neighbours.argtypes = [i64, pd, d, d, i32, i64, pi64, pi64, pi64, pi32, d, pi64, i64]
        L.p3t_oracle_neighbours_sweep.restype = None
        L.p3t_oracle_neighbours_sweep.argtypes = [i64, pd, d, d, i32, pi64, pi64, pi64, pi32]
        L.p3t_oracle_tree_build.restype = vp
        L.p3t_oracle_tree_build.argtypes = [i64, pd, pd, i32, i32]
        L.p3t_oracle_tree_free.restype = None; L.p3t_oracle_tree_free.argtypes = [vp]
        L.p3t_oracle_tree_nnodes.restype = i64; L.p3t_oracle_tree_nnodes.argtypes = [vp]
        L.p3t_oracle_tree_node.restype = None; L.p3t_oracle_tree_node.argtypes = [vp, i64, pd]
        L.p3t_oracle_tree_perm.restype = None; L.p3t_oracle_tree_perm.argtypes = [vp, pi32]
        L.p3t_oracle_tree_walk.restype = None
        L.p3t_oracle_tree_walk.argtypes = [vp, d, d, d, d, d, i32, i64, pi64, pd, pd, pd, pi64, pi32, i64, pi64]
        L.p3t_oracle_num_threads.restype = i32
        L.p3t_oracle_dKdx.restype = d; L.p3t_oracle_dKdx.argtypes = [d]
        L.p3t_oracle_hard.restype = None
        L.p3t_oracle_hard.argtypes = [i64, pd, pd, pd, d, d, d, i64, pi64, pd, pd, pd]
        L.p3t_oracle_hermite.restype = i64
        L.p3t_oracle_hermite.argtypes = [i64, pd, pd, pd, d, d, d, pi64, pi32, d, i32, d, d, d, i64, pi64, pi64]
        pu8 = C.POINTER(C.c_uint8)
        L.p3t_oracle_direct_classes.restype = None
        L.p3t_oracle_direct_classes.argtypes = [i64, pd, pd, pu8, pd, i64, pi64, pd, pd, pd, pd]
        L.p3t_oracle_neighbours_classes.restype = i64
        L.p3t_oracle_neighbours_classes.argtypes = [i64, pd, pu8, pd, i64, pi64, pi64, pi64, pi32, d, pi64, i64]
        L.p3t_oracle_hard_classes.restype = None
        L.p3t_oracle_hard_classes.argtypes = [i64, pd, pd, pd, pu8, pd, i64, pi64, pd, pd, pd]
        L.p3t_oracle_tree_walk_classes.restype = None
        L.p3t_oracle_tree_walk_classes.argtypes = [vp, pu8, pd, d, i32, i64, pi64, pd, pu8, pd, pd, pi64, pi32, i64, pi64]
        L.p3t_oracle_hermite_classes.restype = i64
        L.p3t_oracle_hermite_classes.argtypes = [i64, pd, pd, pd, pu8, pd, pi64, pi32, d, i32, pd, pd, pd, i64, pi64, pi64]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().p3t_oracle_num_threads())


def _f64(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _subset(subset):
    if subset is None:
        return None
    return np.ascontiguousarray(np.asarray(subset), dtype=np.int64)


# ---------------------------------------------------------------- O1 -------
def K(x):
    """Eq. 12."""
    f = lib().p3t_oracle_K
    return np.vectorize(lambda v: f(float(v)), otypes=[np.float64])(x)


def W(y, gamma):
    """Eq. 16-17, reading A1."""
    f = lib().p3t_oracle_W
    return np.vectorize(lambda v: f(float(v), float(gamma)), otypes=[np.float64])(y)


def G(y, gamma):
    f = lib().p3t_oracle_G
    return np.vectorize(lambda v: f(float(v), float(gamma)), otypes=[np.float64])(y)


def Cin(gamma):
    return float(lib().p3t_oracle_Cin(float(gamma)))


def pair_weights(s, r_in, r_out):
    """(K, W) for softened separation s (Eq. 12-17 with Eq. 13-15's x, y, gamma)."""
    k, w = C.c_double(), C.c_double()
    lib().p3t_oracle_pair_weights(float(s), float(r_in), float(r_out), C.byref(k), C.byref(w))
    return k.value, w.value


# ---------------------------------------------------------------- O2 -------
def direct(mass, pos, eps, r_in, r_out, subset=None, hard=False):
    """Direct-sum soft acceleration [ns,3] and potential [ns] (Eq. 6, 8).

    hard=True also returns the complementary (1-K), (1-W) sums (Eq. 5, 7).
    """
    m, q = _f64(mass), _f64(pos).reshape(-1, 3)
    n = m.shape[0]
    sub = _subset(subset)
    ns = n if sub is None else sub.shape[0]
    a_s, p_s = np.empty((ns, 3)), np.empty(ns)
    a_h = np.empty((ns, 3)) if hard else None
    p_h = np.empty(ns) if hard else None
    d = C.c_double
    lib().p3t_oracle_direct(n, _p(m, d), _p(q, d), float(eps), float(r_in), float(r_out), ns,
                            _p(sub, C.c_int64), _p(a_s, d), _p(p_s, d), _p(a_h, d), _p(p_h, d))
    return (a_s, p_s, a_h, p_h) if hard else (a_s, p_s)


# ---------------------------------------------------------------- O6 -------
def dKdx(x):
    """dK/dx of Eq. 12: 140 x^3 (1-x)^3 on [0, 1)."""
    return lib().p3t_oracle_dKdx(float(x))


def hard(mass, pos, vel, eps, r_in, r_out, subset=None):
    """Hard acceleration, its time derivative (jerk) and hard potential per unit mass over all j != i
    (Eq. 7 / Eq. 5; the Hermite part's inputs, L147).  Returns (acc[ns,3], jerk[ns,3], pot[ns])."""
    m, q, v = _f64(mass), _f64(pos).reshape(-1, 3), _f64(vel).reshape(-1, 3)
    n = m.shape[0]
    sub = _subset(subset)
    ns = n if sub is None else sub.shape[0]
    a, j, p = np.empty((ns, 3)), np.empty((ns, 3)), np.empty(ns)
    d = C.c_double
    lib().p3t_oracle_hard(n, _p(m, d), _p(q, d), _p(v, d), float(eps), float(r_in), float(r_out), ns,
                          _p(sub, C.c_int64), _p(a, d), _p(j, d), _p(p, d))
    return a, j, p


# ---------------------------------------------------------------- O7 -------
def hermite(mass, pos, vel, eps, r_in, r_out, offset, nbr, T, log2_div=2, eta=0.1, eta_s=0.01, a0=0.0,
            max_blocks=1 << 22):
    """One soft step T under H_hard (procedure step 3, L147): drift of the particles with empty lists, fourth-order
    Hermite with block timesteps (Eq. 18-20) over the given neighbour lists for the others.
    Returns (pos, vel, info) with info = dict(blocks, nstep[n], floor_hits); raises when max_blocks is exceeded."""
    m = _f64(mass)
    q, v = _f64(pos).reshape(-1, 3).copy(), _f64(vel).reshape(-1, 3).copy()
    n = m.shape[0]
    off = np.ascontiguousarray(offset, dtype=np.int64)
    lst = np.ascontiguousarray(nbr, dtype=np.int32)
    if lst.size == 0:
        lst = np.zeros(1, dtype=np.int32)
    nstep = np.zeros(n, dtype=np.int64)
    fh = np.zeros(1, dtype=np.int64)
    d, i64 = C.c_double, C.c_int64
    nb = lib().p3t_oracle_hermite(n, _p(m, d), _p(q, d), _p(v, d), float(eps), float(r_in), float(r_out),
                                  _p(off, i64), _p(lst, C.c_int32), float(T), int(log2_div), float(eta),
                                  float(eta_s), float(a0), int(max_blocks), _p(nstep, i64), _p(fh, i64))
    if nb < 0:
        raise RuntimeError(f"hermite: more than {max_blocks} blocks (a0 = {a0})")
    return q, v, dict(blocks=int(nb), nstep=nstep, floor_hits=int(fh[0]))


def p3t_step(mass, pos, vel, acc_soft, offset, nbr, eps, r_in, r_out, h, T, log2_div=2, eta=0.1, eta_s=0.01, a0=0.0):
    """One step of the scheme (L142-153) with the soft force by direct sum (O2) and exact lists (O3):
    kick T/2 with acc_soft(t), hard integration over T with the lists made at t, soft force and lists at t + T,
    kick T/2.  Returns (pos, vel, acc_soft, offset, nbr, info)."""
    v = _f64(vel).reshape(-1, 3) + 0.5 * T * _f64(acc_soft).reshape(-1, 3)
    q, v, info = hermite(mass, pos, v, eps, r_in, r_out, offset, nbr, T, log2_div, eta, eta_s, a0)
    a, _ = direct(mass, q, eps, r_in, r_out)
    off, lst, _ = neighbours(q, eps, h)
    v = v + 0.5 * T * a
    return q, v, a, off, lst, info


# ---------------------------------------------------------------- O3 -------
def neighbours(pos, eps, h, subset=None, plain=False, band=1e-6):
    """Exact neighbour sets by brute force.

    Returns (offset[ns+1], nbr[total] ascending per list, band_pairs[nb,2]) where
    band_pairs holds (k, j) with |s_kj/h - 1| < band (k indexes the subset).
    """
    q = _f64(pos).reshape(-1, 3)
    n = q.shape[0]
    sub = _subset(subset)
    ns = n if sub is None else sub.shape[0]
    count = np.zeros(ns, dtype=np.int64)
    d, i64 = C.c_double, C.c_int64
    L = lib()
    nb = L.p3t_oracle_neighbours(n, _p(q, d), float(eps), float(h), int(plain), ns, _p(sub, i64),
                                 _p(count, i64), None, None, float(band), None, 0)
    offset = np.zeros(ns + 1, dtype=np.int64)
    np.cumsum(count, out=offset[1:])
    lst = np.empty(max(int(offset[-1]), 1), dtype=np.int32)
    bp = np.empty((max(int(nb), 1), 2), dtype=np.int64)
    L.p3t_oracle_neighbours(n, _p(q, d), float(eps), float(h), int(plain), ns, _p(sub, i64),
                            None, _p(offset, i64), _p(lst, C.c_int32), float(band), _p(bp, i64), int(nb))
    return offset, lst[: int(offset[-1])], bp[: int(nb)]


def neighbours_sweep(pos, eps, h, plain=False):
    """Exact neighbour sets of all particles by sort-and-sweep along x."""
    q = _f64(pos).reshape(-1, 3)
    n = q.shape[0]
    order = np.ascontiguousarray(np.argsort(q[:, 0], kind="stable"), dtype=np.int64)
    count = np.zeros(n, dtype=np.int64)
    d, i64 = C.c_double, C.c_int64
    L = lib()
    L.p3t_oracle_neighbours_sweep(n, _p(q, d), float(eps), float(h), int(plain), _p(order, i64),
                                  _p(count, i64), None, None)
    offset = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(count, out=offset[1:])
    lst = np.empty(max(int(offset[-1]), 1), dtype=np.int32)
    L.p3t_oracle_neighbours_sweep(n, _p(q, d), float(eps), float(h), int(plain), _p(order, i64),
                                  None, _p(offset, i64), _p(lst, C.c_int32))
    return offset, lst[: int(offset[-1])]


# ---------------------------------------------------------------- O8 -------
def pair_table(eps, r_in, r_out, h, r_in_bf, r_out_bf, h_bf, eps_bb=0.0, eps_bf=None):
    """tab[3][4] = (eps, r_in, r_cut, h) for the kinds FS-FS, BH-FS, BH-BH of section 3.2.2.1 (L287); BH-BH is not
    split (r_cut = inf).  eps_bf defaults to eps (the paper uses one softening for FS-FS and FS-SMBH)."""
    return np.array([[eps, r_in, r_out, h],
                     [eps if eps_bf is None else eps_bf, r_in_bf, r_out_bf, h_bf],
                     [eps_bb, np.inf, np.inf, np.inf]], dtype=np.float64)


def _cls(classes):
    return np.ascontiguousarray(np.asarray(classes), dtype=np.uint8)


def direct_classes(mass, pos, classes, tab, subset=None, hard=False):
    """O2 with a class per body and cutoffs per kind of pair (L287)."""
    m, q, c, t = _f64(mass), _f64(pos).reshape(-1, 3), _cls(classes), _f64(tab)
    n = m.shape[0]
    sub = _subset(subset)
    ns = n if sub is None else sub.shape[0]
    a_s, p_s = np.empty((ns, 3)), np.empty(ns)
    a_h = np.empty((ns, 3)) if hard else None
    p_h = np.empty(ns) if hard else None
    d = C.c_double
    lib().p3t_oracle_direct_classes(n, _p(m, d), _p(q, d), _p(c, C.c_uint8), _p(t, d), ns, _p(sub, C.c_int64),
                                    _p(a_s, d), _p(p_s, d), _p(a_h, d), _p(p_h, d))
    return (a_s, p_s, a_h, p_h) if hard else (a_s, p_s)


def neighbours_classes(pos, classes, tab, subset=None, band=1e-6):
    """O3 with the pair's own h; pairs of an unsplit kind are always neighbours."""
    q, c, t = _f64(pos).reshape(-1, 3), _cls(classes), _f64(tab)
    n = q.shape[0]
    sub = _subset(subset)
    ns = n if sub is None else sub.shape[0]
    count = np.zeros(ns, dtype=np.int64)
    d, i64 = C.c_double, C.c_int64
    L = lib()
    nb = L.p3t_oracle_neighbours_classes(n, _p(q, d), _p(c, C.c_uint8), _p(t, d), ns, _p(sub, i64),
                                         _p(count, i64), None, None, float(band), None, 0)
    offset = np.zeros(ns + 1, dtype=np.int64)
    np.cumsum(count, out=offset[1:])
    lst = np.empty(max(int(offset[-1]), 1), dtype=np.int32)
    bp = np.empty((max(int(nb), 1), 2), dtype=np.int64)
    L.p3t_oracle_neighbours_classes(n, _p(q, d), _p(c, C.c_uint8), _p(t, d), ns, _p(sub, i64),
                                    None, _p(offset, i64), _p(lst, C.c_int32), float(band), _p(bp, i64), int(nb))
    return offset, lst[: int(offset[-1])], bp[: int(nb)]


def hard_classes(mass, pos, vel, classes, tab, subset=None):
    """O6 with classes: (acc, jerk, pot) of the hard part over all j != i."""
    m, q, v, c, t = _f64(mass), _f64(pos).reshape(-1, 3), _f64(vel).reshape(-1, 3), _cls(classes), _f64(tab)
    n = m.shape[0]
    sub = _subset(subset)
    ns = n if sub is None else sub.shape[0]
    a, j, p = np.empty((ns, 3)), np.empty((ns, 3)), np.empty(ns)
    d = C.c_double
    lib().p3t_oracle_hard_classes(n, _p(m, d), _p(q, d), _p(v, d), _p(c, C.c_uint8), _p(t, d), ns,
                                  _p(sub, C.c_int64), _p(a, d), _p(j, d), _p(p, d))
    return a, j, p


def hermite_classes(mass, pos, vel, classes, tab, offset, nbr, T, log2_div=2, eta=(0.1, 0.03), eta_s=(0.01, 0.003),
                    a0=(0.0, 0.0), max_blocks=1 << 22):
    """O7 with pair classes (L287): eta, eta_s, a0 are (field star, black hole) pairs.  Returns (pos, vel, info)."""
    m = _f64(mass)
    q, v = _f64(pos).reshape(-1, 3).copy(), _f64(vel).reshape(-1, 3).copy()
    n = m.shape[0]
    c, t = _cls(classes), _f64(tab)
    off = np.ascontiguousarray(offset, dtype=np.int64)
    lst = np.ascontiguousarray(nbr, dtype=np.int32)
    if lst.size == 0:
        lst = np.zeros(1, dtype=np.int32)
    nstep = np.zeros(n, dtype=np.int64)
    fh = np.zeros(1, dtype=np.int64)
    e, es, aa = _f64(eta), _f64(eta_s), _f64(a0)
    d, i64 = C.c_double, C.c_int64
    nb = lib().p3t_oracle_hermite_classes(n, _p(m, d), _p(q, d), _p(v, d), _p(c, C.c_uint8), _p(t, d), _p(off, i64),
                                          _p(lst, C.c_int32), float(T), int(log2_div), _p(e, d), _p(es, d), _p(aa, d),
                                          int(max_blocks), _p(nstep, i64), _p(fh, i64))
    if nb < 0:
        raise RuntimeError(f"hermite_classes: more than {max_blocks} blocks")
    return q, v, dict(blocks=int(nb), nstep=nstep, floor_hits=int(fh[0]))


# ---------------------------------------------------------------- O4 -------
class Tree:
    """Pointer-based Barnes-Hut octree with monopole + quadrupole moments (L138)."""

    NODE_FIELDS = 32

    def __init__(self, mass, pos, nleaf=16, max_depth=21):
        self.m, self.q = _f64(mass), _f64(pos).reshape(-1, 3)
        self.n = self.m.shape[0]
        d = C.c_double
        self._h = lib().p3t_oracle_tree_build(self.n, _p(self.m, d), _p(self.q, d), int(nleaf), int(max_depth))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().p3t_oracle_tree_free(self._h)
            self._h = None

    @property
    def nnodes(self):
        return int(lib().p3t_oracle_tree_nnodes(self._h))

    def nodes(self):
        """Structured view of every node (for the moment / topology pins)."""
        out = np.empty((self.nnodes, self.NODE_FIELDS))
        row = np.empty(self.NODE_FIELDS)
        for k in range(self.nnodes):
            lib().p3t_oracle_tree_node(self._h, k, _p(row, C.c_double))
            out[k] = row
        return dict(g=out[:, 0:3], side=out[:, 3], M=out[:, 4], c=out[:, 5:8], Q=out[:, 8:14],
                    bmin=out[:, 14:17], bmax=out[:, 17:20], first=out[:, 20].astype(np.int64),
                    count=out[:, 21].astype(np.int64), leaf=out[:, 22].astype(bool),
                    level=out[:, 23].astype(np.int64), child=out[:, 24:32].astype(np.int64))

    def perm(self):
        p = np.empty(self.n, dtype=np.int32)
        lib().p3t_oracle_tree_perm(self._h, _p(p, C.c_int32))
        return p

    def walk(self, eps, theta, r_in, r_out, h, subset=None, box=None, use_quad=True, nbr_stride=0):
        """Returns dict(acc[ns,3], pot[ns], n_pp[ns], n_pc[ns], nbr_count[ns], nbr[ns,stride])."""
        sub = _subset(subset)
        ns = self.n if sub is None else sub.shape[0]
        acc, pot = np.empty((ns, 3)), np.empty(ns)
        counts = np.zeros((ns, 2), dtype=np.int64)
        nbr_count = np.zeros(ns, dtype=np.int64)
        nbr = np.full((ns, nbr_stride), -1, dtype=np.int32) if nbr_stride else None
        bx = None if box is None else _f64(box).reshape(ns, 6)
        d, i64 = C.c_double, C.c_int64
        lib().p3t_oracle_tree_walk(self._h, float(eps), float(theta), float(r_in), float(r_out), float(h),
                                   int(use_quad), ns, _p(sub, i64), _p(bx, d), _p(acc, d), _p(pot, d),
                                   _p(counts, i64), _p(nbr, C.c_int32), int(nbr_stride), _p(nbr_count, i64))
        return dict(acc=acc, pot=pot, n_pp=counts[:, 0], n_pc=counts[:, 1], nbr_count=nbr_count, nbr=nbr)

    def walk_classes(self, classes, tab, theta, subset=None, box=None, box_mask=None, use_quad=True, nbr_stride=0):
        """O4 with classes (L287): same outputs as walk()."""
        sub = _subset(subset)
        ns = self.n if sub is None else sub.shape[0]
        acc, pot = np.empty((ns, 3)), np.empty(ns)
        counts = np.zeros((ns, 2), dtype=np.int64)
        nbr_count = np.zeros(ns, dtype=np.int64)
        nbr = np.full((ns, nbr_stride), -1, dtype=np.int32) if nbr_stride else None
        bx = None if box is None else _f64(box).reshape(ns, 6)
        bm = None if box_mask is None else _cls(box_mask)
        c, t = _cls(classes), _f64(tab)
        d, i64 = C.c_double, C.c_int64
        lib().p3t_oracle_tree_walk_classes(self._h, _p(c, C.c_uint8), _p(t, d), float(theta), int(use_quad), ns,
                                           _p(sub, i64), _p(bx, d), _p(bm, C.c_uint8), _p(acc, d), _p(pot, d),
                                           _p(counts, i64), _p(nbr, C.c_int32), int(nbr_stride), _p(nbr_count, i64))
        return dict(acc=acc, pot=pot, n_pp=counts[:, 0], n_pc=counts[:, 1], nbr_count=nbr_count, nbr=nbr)
