"""Helpers shared by the GPU parity tests (comparison logic only; no method arithmetic)."""
import numpy as np


def widen(cfg):
    """fp32 inputs widened to fp64: what the oracle consumes."""
    return cfg["mass"].astype(np.float64), cfg["pos"].astype(np.float64)


def rel_err(a, ref):
    return np.linalg.norm(a - ref, axis=1) / np.linalg.norm(ref, axis=1)


def csr_sets(offset, nbr, rows=None):
    rows = range(len(offset) - 1) if rows is None else rows
    return [set(nbr[int(offset[i]):int(offset[i + 1])].tolist()) for i in rows]


def assert_same_neighbour_sets(gpu_sets, ora_sets, band_pairs, ids=None):
    """Set-identical lists, except pairs inside the 1e-6 band around h (north_star)."""
    band = {}
    for k, j in np.asarray(band_pairs).reshape(-1, 2):
        band.setdefault(int(k), set()).add(int(j))
    bad = []
    for k, (g, o) in enumerate(zip(gpu_sets, ora_sets)):
        diff = (g ^ o) - band.get(k, set())
        if diff:
            bad.append((k if ids is None else int(ids[k]), sorted(diff)[:5]))
    assert not bad, f"{len(bad)} lists differ outside the band, e.g. {bad[:5]}"
