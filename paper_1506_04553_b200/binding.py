"""Thin Python front end of the C-ABI library (include/p3t.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libp3t.so.  torch supplies
device memory (the workspace and optional device-side inputs/outputs) and the
stream.  There is no CPU fallback: importing this module without the built
library raises ImportError.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libp3t.so")

if not os.path.exists(_LIBPATH):
    raise ImportError(
        f"{_LIBPATH} is missing: build it with `python -m paper_1506_04553_b200.build` "
        "(there is no CPU fallback for the soft-force path)")

_lib = C.CDLL(_LIBPATH)

OK, EINVAL, ESTATE, ENOMEM, ECAPACITY, ECUDA, ELIMIT = 0, -1, -2, -3, -4, -5, -6
_STATUS = {0: "P3T_OK", -1: "P3T_EINVAL", -2: "P3T_ESTATE", -3: "P3T_ENOMEM", -4: "P3T_ECAPACITY", -5: "P3T_ECUDA", -6: "P3T_ELIMIT"}

# names of include/p3t.h's exported entry points (tests check that each resolves)
SYMBOLS = [
    "p3t_workspace_bytes", "p3t_create", "p3t_destroy", "p3t_set_params", "p3t_set_tree_params",
    "p3t_set_pair_classes", "p3t_set_key_curve", "p3t_set_sort_passes", "p3t_hilbert_state_tables", "p3t_set_group_merge_levels", "p3t_set_walk_mode", "p3t_set_shard", "p3t_get_shard_record", "p3t_put_shard_classes", "p3t_load_particles", "p3t_build_tree", "p3t_set_tree_reuse", "p3t_refit_tree", "p3t_eval_soft", "p3t_eval_direct", "p3t_direct_static", "p3t_direct_static_last_error", "p3t_eval_hard",
    "p3t_hermite_step", "p3t_step", "p3t_set_hermite_cluster_max", "p3t_set_hermite_class_params",
    "p3t_get_acc_pot", "p3t_get_neighbour_counts", "p3t_get_neighbours", "p3t_get_stats", "p3t_synchronize",
    "p3t_last_error", "p3t_array_info", "p3t_copy_array", "p3t_measure_fp32_peak", "p3t_measure_latency",
]

ARRAYS = dict(root_cube=(0, np.float32, 1), keys=(1, np.uint64, 1), sorted_idx=(2, np.uint32, 1),
              bodies=(3, np.float32, 4), cell_mac=(4, np.float32, 4), cell_mom0=(5, np.float32, 4),
              cell_mom1=(6, np.float32, 4), cell_meta=(7, np.uint32, 2), cell_level=(8, np.uint8, 1),
              cell_start=(9, np.uint32, 1), cell_parent=(10, np.uint32, 1), group_start=(11, np.uint32, 1), group_stats=(14, np.uint32, 4), group_order=(15, np.uint32, 1),
              cell_bmin=(12, np.float32, 4), cell_bmax=(13, np.float32, 4))


class Stats(C.Structure):
    _fields_ = [("n", C.c_uint64), ("n_pp", C.c_uint64), ("n_pc", C.c_uint64), ("n_near", C.c_uint64),
                ("n_neighbours", C.c_uint64), ("n_cells", C.c_uint32), ("n_leaves", C.c_uint32),
                ("n_groups", C.c_uint32), ("depth", C.c_uint32), ("max_list", C.c_uint32),
                ("sort_passes", C.c_uint32), ("ms_sort", C.c_float), ("ms_build", C.c_float),
                ("ms_moments", C.c_float), ("ms_walk", C.c_float), ("ms_nbr", C.c_float), ("ms_hard", C.c_float), ("ms_pack", C.c_float),
                ("tree_refits", C.c_uint32), ("n_stray", C.c_uint32), ("walk_parts", C.c_uint32), ("sort_max_run", C.c_uint32)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class HermiteInfo(C.Structure):
    _fields_ = [("n_nonisolated", C.c_uint64), ("n_blocks", C.c_uint64), ("n_steps", C.c_uint64),
                ("floor_hits", C.c_uint64), ("n_components", C.c_uint64), ("max_component", C.c_uint64), ("ms", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def _sig():
    vp, sz, i, f = C.c_void_p, C.c_size_t, C.c_int, C.c_float
    L = _lib
    L.p3t_workspace_bytes.restype = sz; L.p3t_workspace_bytes.argtypes = [sz, i, sz]
    L.p3t_create.restype = i; L.p3t_create.argtypes = [C.POINTER(vp), i, sz, i, vp, sz, sz, vp]
    L.p3t_destroy.restype = i; L.p3t_destroy.argtypes = [vp]
    L.p3t_set_params.restype = i; L.p3t_set_params.argtypes = [vp, f, f, f, f, f]
    L.p3t_set_tree_params.restype = i; L.p3t_set_tree_params.argtypes = [vp, i, i]
    L.p3t_set_pair_classes.restype = i; L.p3t_set_pair_classes.argtypes = [vp, sz, vp, i, f, f, f, f]
    L.p3t_set_group_merge_levels.restype = i; L.p3t_set_group_merge_levels.argtypes = [vp, i]
    L.p3t_set_sort_passes.restype = i; L.p3t_set_sort_passes.argtypes = [vp, i]
    L.p3t_direct_static.restype = i
    L.p3t_direct_static.argtypes = [i, vp, C.c_size_t, vp, vp, C.c_float, C.c_float, C.c_float, C.c_float, vp, vp, vp, vp]
    L.p3t_direct_static_last_error.restype = C.c_char_p; L.p3t_direct_static_last_error.argtypes = []
    L.p3t_set_key_curve.restype = i; L.p3t_set_key_curve.argtypes = [vp, i]
    L.p3t_hilbert_state_tables.restype = i; L.p3t_hilbert_state_tables.argtypes = [vp, sz]
    L.p3t_set_walk_mode.restype = i; L.p3t_set_walk_mode.argtypes = [vp, i]
    L.p3t_set_hermite_cluster_max.restype = i; L.p3t_set_hermite_cluster_max.argtypes = [vp, i]
    L.p3t_set_hermite_class_params.restype = i; L.p3t_set_hermite_class_params.argtypes = [vp, C.c_double, C.c_double, C.c_double]
    L.p3t_set_shard.restype = i; L.p3t_set_shard.argtypes = [vp, i, i]
    L.p3t_get_shard_record.restype = i; L.p3t_get_shard_record.argtypes = [vp, vp]
    L.p3t_put_shard_classes.restype = i; L.p3t_put_shard_classes.argtypes = [vp, vp]
    L.p3t_load_particles.restype = i; L.p3t_load_particles.argtypes = [vp, sz, vp, vp, i]
    L.p3t_build_tree.restype = i; L.p3t_build_tree.argtypes = [vp]
    L.p3t_eval_soft.restype = i; L.p3t_eval_soft.argtypes = [vp]
    L.p3t_refit_tree.restype = i; L.p3t_refit_tree.argtypes = [vp]
    L.p3t_set_tree_reuse.restype = i; L.p3t_set_tree_reuse.argtypes = [vp, i, f, f]
    L.p3t_eval_direct.restype = i; L.p3t_eval_direct.argtypes = [vp, vp, sz, i]
    L.p3t_eval_hard.restype = i; L.p3t_eval_hard.argtypes = [vp, vp, vp, vp, vp, i]
    d, ll = C.c_double, C.c_longlong
    L.p3t_hermite_step.restype = i; L.p3t_hermite_step.argtypes = [vp, vp, vp, d, i, d, d, d, ll, i, C.POINTER(HermiteInfo)]
    L.p3t_step.restype = i; L.p3t_step.argtypes = [vp, vp, vp, vp, d, i, d, d, d, ll, i, C.POINTER(HermiteInfo)]
    L.p3t_get_acc_pot.restype = i; L.p3t_get_acc_pot.argtypes = [vp, vp, vp, i]
    L.p3t_get_neighbour_counts.restype = i; L.p3t_get_neighbour_counts.argtypes = [vp, vp, C.POINTER(C.c_uint64), i]
    L.p3t_get_neighbours.restype = i; L.p3t_get_neighbours.argtypes = [vp, vp, vp, sz, i]
    L.p3t_get_stats.restype = i; L.p3t_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.p3t_synchronize.restype = i; L.p3t_synchronize.argtypes = [vp]
    L.p3t_last_error.restype = C.c_char_p; L.p3t_last_error.argtypes = [vp]
    L.p3t_array_info.restype = i; L.p3t_array_info.argtypes = [vp, i, C.POINTER(sz), C.POINTER(sz)]
    L.p3t_copy_array.restype = i; L.p3t_copy_array.argtypes = [vp, i, vp, sz, i]
    L.p3t_measure_latency.restype = i; L.p3t_measure_latency.argtypes = [vp, i, i, C.POINTER(C.c_double)]
    L.p3t_measure_fp32_peak.restype = i
    L.p3t_measure_fp32_peak.argtypes = [vp, i, i, C.POINTER(C.c_double), C.POINTER(C.c_float)]


_sig()


class P3TError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def hilbert_state_tables():
    """The state tables the key kernel uses for Peano-Hilbert keys (host only, no GPU needed): uint32[24 * 64 + 24 * 8]."""
    tab = np.zeros(24 * 64 + 24 * 8, dtype=np.uint32)
    st = _lib.p3t_hilbert_state_tables(tab.ctypes.data, tab.size)
    if st != OK:
        raise P3TError(st, "the tables derived from the transform are inconsistent")
    return tab


def p3t_workspace_bytes(max_n, key_bits=63, nbr_capacity=0):
    return int(_lib.p3t_workspace_bytes(max_n, key_bits, nbr_capacity))


STATIC_MAX_N = 65536     # P3T_STATIC_MAX_N of include/p3t.h


def direct_static(mass, pos, eps, r_in, r_out, r_search, acc, pot, nbr_count=None, info=None, stream=None):
    """p3t_direct_static: brute-force soft force with the library's static scratch (no context, nothing allocated).
    All arrays are contiguous CUDA tensors of the caller (mass [n], pos [n, 3], acc [n, 3], pot [n] float32; nbr_count [n]
    int32, info [2] int64, both optional) on one device.  Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    for t, dt in ((mass, torch.float32), (pos, torch.float32), (acc, torch.float32), (pot, torch.float32)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise TypeError("direct_static takes contiguous float32 CUDA tensors")
    for t, dt in ((nbr_count, torch.int32), (info, torch.int64)):
        if t is not None and not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise TypeError("nbr_count must be an int32, info an int64 CUDA tensor")
    n = mass.shape[0]
    if pos.numel() != 3 * n or acc.numel() != 3 * n or pot.numel() != n or (nbr_count is not None and nbr_count.numel() != n) \
            or (info is not None and info.numel() < 2):
        raise ValueError("direct_static: array sizes do not fit n")
    dev = mass.device.index
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    st = _lib.p3t_direct_static(dev, s.cuda_stream, n, mass.data_ptr(), pos.data_ptr(), float(eps), float(r_in), float(r_out),
                                float(r_search), acc.data_ptr(), pot.data_ptr(),
                                nbr_count.data_ptr() if nbr_count is not None else None, info.data_ptr() if info is not None else None)
    if st != OK:
        raise P3TError(st, _lib.p3t_direct_static_last_error().decode())


def _ptr(x):
    """Raw address of a numpy array (host) or torch tensor (device); None -> NULL."""
    if x is None:
        return None, 0
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data, 0
    import torch
    assert isinstance(x, torch.Tensor) and x.is_contiguous()
    return x.data_ptr(), int(x.is_cuda)


class P3T:
    """One soft-force context (one GPU, one stream).  Method names follow the C ABI."""

    def __init__(self, max_n, key_bits=63, nbr_capacity=None, device=0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1506_04553_b200 needs a CUDA device; there is no CPU path")
        self.torch = torch
        self.device = device
        self.max_n = int(max_n)
        self.nbr_capacity = int(nbr_capacity if nbr_capacity is not None else max(4 * max_n, 1 << 16))
        nbytes = p3t_workspace_bytes(self.max_n, key_bits, self.nbr_capacity)
        if nbytes == 0:
            raise P3TError(EINVAL, "invalid max_n / key_bits")
        with torch.cuda.device(device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=f"cuda:{device}")
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            self._stream = stream if stream is not None else torch.cuda.current_stream(device)
        h = C.c_void_p()
        st = _lib.p3t_create(C.byref(h), device, self.max_n, key_bits, self._ws_ptr, nbytes, self.nbr_capacity,
                             self._stream.cuda_stream)
        if st != OK:
            raise P3TError(st, "p3t_create failed")
        self._h = h
        self.n = 0

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, st):
        if st != OK:
            raise P3TError(st, _lib.p3t_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            _lib.p3t_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the C ABI, one method per entry point --------------------------------------------------------
    def set_params(self, eps, theta, r_in, r_out, r_search):
        self._check(_lib.p3t_set_params(self._h, eps, theta, r_in, r_out, r_search))

    def set_tree_params(self, nleaf=16, ngroup=64):
        self._check(_lib.p3t_set_tree_params(self._h, nleaf, ngroup))

    def set_pair_classes(self, classes, r_in_bf=0.0, r_out_bf=1.0, r_search_bf=1.0, eps_bb=0.0):
        """classes: uint8 [n] numpy (host) or CUDA tensor, 0 field star / 1 black hole; None switches classes off."""
        if classes is None:
            self._check(_lib.p3t_set_pair_classes(self._h, 0, None, 0, 0.0, 1.0, 1.0, 0.0))
            return
        pc, dc = _ptr(classes)
        if str(classes.dtype).split(".")[-1] != "uint8":
            raise P3TError(EINVAL, "classes must be uint8")
        self._check(_lib.p3t_set_pair_classes(self._h, int(classes.shape[0]), pc, dc, r_in_bf, r_out_bf, r_search_bf, eps_bb))

    def set_key_curve(self, curve):
        """'morton' / 0 or 'hilbert' / 1 (default)."""
        c = {"morton": 0, "hilbert": 1}.get(curve, curve)
        self._check(_lib.p3t_set_key_curve(self._h, int(c)))

    def set_sort_passes(self, passes):
        self._check(_lib.p3t_set_sort_passes(self._h, int(passes)))

    def set_group_merge_levels(self, levels):
        self._check(_lib.p3t_set_group_merge_levels(self._h, levels))

    def set_walk_mode(self, mode):
        self._check(_lib.p3t_set_walk_mode(self._h, mode))

    def set_shard(self, rank, world):
        self._check(_lib.p3t_set_shard(self._h, rank, world))

    def get_shard_record(self, rec=None):
        """float32 CUDA tensor [n, 5]: (a, phi, cost class + 1) of the particles this shard produced, zeros elsewhere."""
        t = self.torch
        if rec is None:
            rec = t.empty((self.n, 5), dtype=t.float32, device=f"cuda:{self.device}")
        assert rec.is_cuda and rec.is_contiguous() and rec.numel() == 5 * self.n and rec.dtype == t.float32
        self._check(_lib.p3t_get_shard_record(self._h, rec.data_ptr()))
        return rec

    def put_shard_classes(self, rec):
        assert rec.is_cuda and rec.is_contiguous() and rec.numel() == 5 * self.n
        self._check(_lib.p3t_put_shard_classes(self._h, rec.data_ptr()))

    def load_particles(self, mass, pos):
        """mass[n], pos[n,3] (or [3n]): float32 numpy arrays (host) or CUDA tensors (device)."""
        pm, dm = _ptr(mass)
        pp, dp = _ptr(pos)
        if dm != dp:
            raise P3TError(EINVAL, "mass and pos must both be host or both be device")
        n = int(mass.shape[0])
        if str(mass.dtype).split(".")[-1] != "float32" or str(pos.dtype).split(".")[-1] != "float32":
            raise P3TError(EINVAL, "mass and pos must be float32")
        if int(np.prod(pos.shape)) != 3 * n:
            raise P3TError(EINVAL, "pos must hold 3 n values")
        self._check(_lib.p3t_load_particles(self._h, n, pm, pp, dm))
        self.n = n
        self._keep = (mass, pos)   # keep inputs alive until the stream has consumed them

    def build_tree(self):
        self._check(_lib.p3t_build_tree(self._h))

    def eval_soft(self):
        self._check(_lib.p3t_eval_soft(self._h))

    def set_tree_reuse(self, max_refits, stray_dist=0.5, max_stray_fraction=0.02):
        self._check(_lib.p3t_set_tree_reuse(self._h, int(max_refits), stray_dist, max_stray_fraction))

    def refit_tree(self):
        self._check(_lib.p3t_refit_tree(self._h))

    def eval_direct(self, subset=None):
        if subset is None:
            self._check(_lib.p3t_eval_direct(self._h, None, 0, 0))
        else:
            sub = np.ascontiguousarray(subset, dtype=np.uint32)
            self._check(_lib.p3t_eval_direct(self._h, sub.ctypes.data, sub.shape[0], 0))

    def get_acc_pot(self, on_device=False):
        if on_device:
            t = self.torch
            acc = t.empty((self.n, 3), dtype=t.float32, device=f"cuda:{self.device}")
            pot = t.empty(self.n, dtype=t.float32, device=f"cuda:{self.device}")
            self._check(_lib.p3t_get_acc_pot(self._h, acc.data_ptr(), pot.data_ptr(), 1))
            return acc, pot
        acc = np.empty((self.n, 3), dtype=np.float32)
        pot = np.empty(self.n, dtype=np.float32)
        self._check(_lib.p3t_get_acc_pot(self._h, acc.ctypes.data, pot.ctypes.data, 0))
        return acc, pot

    def get_acc_pot_into(self, acc, pot):
        """Write into caller-provided buffers (numpy or CUDA tensors)."""
        pa, da = _ptr(acc)
        pp, dp = _ptr(pot)
        self._check(_lib.p3t_get_acc_pot(self._h, pa, pp, da if acc is not None else dp))

    def eval_hard(self, vel, acc=None, jerk=None, pot=None):
        """Hard acceleration, jerk and potential from the neighbour lists of the last eval (p3t_eval_hard).
        vel: float32 [n,3] numpy (host) or CUDA tensor.  Host form: returns float64 numpy (acc, jerk, pot).
        Device form: writes the given float64 CUDA tensors (any may be None) and returns them."""
        pv, dv = _ptr(vel)
        if dv:
            pa, _ = _ptr(acc); pj, _ = _ptr(jerk); pp, _ = _ptr(pot)
            self._check(_lib.p3t_eval_hard(self._h, pv, pa, pj, pp, 1))
            return acc, jerk, pot
        a, j, p = np.empty((self.n, 3)), np.empty((self.n, 3)), np.empty(self.n)
        self._check(_lib.p3t_eval_hard(self._h, pv, a.ctypes.data, j.ctypes.data, p.ctypes.data, 0))
        return a, j, p

    def set_hermite_class_params(self, eta_bh=0.0, eta_s_bh=0.0, a0_bh=-1.0):
        self._check(_lib.p3t_set_hermite_class_params(self._h, float(eta_bh), float(eta_s_bh), float(a0_bh)))

    def set_hermite_cluster_max(self, max_members):
        self._check(_lib.p3t_set_hermite_cluster_max(self._h, int(max_members)))

    def hermite_step(self, pos, vel, dt_soft, log2_div=2, eta=0.1, eta_s=0.01, a0=0.0, max_blocks=1 << 22):
        """One soft step under H_hard over the lists of the last eval (p3t_hermite_step): pos, vel float64 [n,3], both
        numpy (host) or both CUDA tensors, advanced IN PLACE.  Returns the statistics as a dict."""
        pp, dp = _ptr(pos)
        pv, dv = _ptr(vel)
        assert dp == dv and pos.dtype == vel.dtype and str(pos.dtype).endswith("float64")
        info = HermiteInfo()
        self._check(_lib.p3t_hermite_step(self._h, pp, pv, float(dt_soft), int(log2_div), float(eta), float(eta_s),
                                          float(a0), int(max_blocks), dp, C.byref(info)))
        return info.as_dict()

    def step(self, mass, pos, vel, dt_soft, log2_div=2, eta=0.1, eta_s=0.01, a0=0.0, max_blocks=1 << 22):
        """One step of the scheme (p3t_step): kick, hard part, soft force at the new time, kick.  mass float32 [n],
        pos, vel float64 [n,3], all numpy or all CUDA tensors; pos and vel are advanced IN PLACE."""
        pm, dm = _ptr(mass)
        pp, dp = _ptr(pos)
        pv, dv = _ptr(vel)
        assert dm == dp == dv and str(pos.dtype).endswith("float64") and str(vel.dtype).endswith("float64")
        assert str(mass.dtype).endswith("float32")
        info = HermiteInfo()
        self._check(_lib.p3t_step(self._h, pm, pp, pv, float(dt_soft), int(log2_div), float(eta), float(eta_s),
                                  float(a0), int(max_blocks), dp, C.byref(info)))
        return info.as_dict()

    def get_neighbour_counts(self):
        count = np.empty(self.n, dtype=np.uint32)
        total = C.c_uint64()
        self._check(_lib.p3t_get_neighbour_counts(self._h, count.ctypes.data, C.byref(total), 0))
        return count, int(total.value)

    def get_neighbours(self, capacity=None):
        """CSR (offset[n+1] uint64, nbr[total] uint32) in user ids; lists ascending."""
        cap = self.nbr_capacity if capacity is None else int(capacity)
        offset = np.empty(self.n + 1, dtype=np.uint64)
        nbr = np.empty(max(cap, 1), dtype=np.uint32)
        self._check(_lib.p3t_get_neighbours(self._h, offset.ctypes.data, nbr.ctypes.data, cap, 0))
        return offset, nbr[: int(offset[-1])]

    def get_neighbours_into(self, offset, nbr):
        """Same, into caller-provided host buffers (e.g. pinned): offset uint64[n+1], nbr uint32[capacity].
        Returns the total number of entries."""
        assert offset.dtype == np.uint64 and offset.size >= self.n + 1 and nbr.dtype == np.uint32
        self._check(_lib.p3t_get_neighbours(self._h, offset.ctypes.data, nbr.ctypes.data, nbr.size, 0))
        return int(offset[self.n])

    def get_stats(self):
        s = Stats()
        self._check(_lib.p3t_get_stats(self._h, C.byref(s)))
        return s.as_dict()

    def synchronize(self):
        self._check(_lib.p3t_synchronize(self._h))

    def measure_fp32_peak(self, packed=True, iters=2048):
        """Pure-FFMA calibration kernel: (TFLOP/s, ms) of the best of four launches.
        packed: 0/False scalar FFMA, 1/True FFMA2, 2-4 the FFMA2 operand-pattern variants of include/p3t.h."""
        tf, ms = C.c_double(), C.c_float()
        self._check(_lib.p3t_measure_fp32_peak(self._h, int(packed), int(iters), C.byref(tf), C.byref(ms)))
        return tf.value, ms.value

    def measure_latency(self, what, iters=2000):
        """ns per dependent step (p3t_measure_latency); scribbles over the workspace: load particles again afterwards."""
        ns = C.c_double()
        self._check(_lib.p3t_measure_latency(self._h, int(what), int(iters), C.byref(ns)))
        self.n = 0
        return ns.value

    def array(self, name):
        """Copy of an intermediate array (a1-a6 inspection), as numpy."""
        which, dtype, width = ARRAYS[name]
        cnt, eb = C.c_size_t(), C.c_size_t()
        self._check(_lib.p3t_array_info(self._h, which, C.byref(cnt), C.byref(eb)))
        nbytes = cnt.value * eb.value
        out = np.empty(nbytes // np.dtype(dtype).itemsize, dtype=dtype)
        self._check(_lib.p3t_copy_array(self._h, which, out.ctypes.data, nbytes, 0))
        return out.reshape(-1, width) if width > 1 else out

    # -- convenience: the whole hot path for one batch -------------------------------------------------
    def soft_force(self, mass, pos):
        """load -> build -> eval; returns nothing (fetch with get_*)."""
        self.load_particles(mass, pos)
        self.build_tree()
        self.eval_soft()
