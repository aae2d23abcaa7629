"""Host logic of the product path: the state tables the key kernel uses for Peano-Hilbert keys (derived by the library
from Skilling's transform, include/p3t.h p3t_hilbert_state_tables), replayed in python on the oracle's quantised
coordinates, give the oracle's keys (oracle/keytree.py hilbert_keys) for both key widths.  No GPU involved."""
import numpy as np
import pytest

from oracle import keytree


@pytest.mark.parametrize("L", [21, 10, 2, 1])
def test_table_walk_reproduces_the_oracles_hilbert_keys(L):
    from paper_1506_04553_b200 import binding

    tab = binding.hilbert_state_tables()
    assert tab.shape == (24 * 64 + 24 * 8,)
    rng = np.random.default_rng(L)
    p = rng.uniform(0, 1, (3000, 3)) ** 1.5
    ref = keytree.hilbert_keys(p, [0, 0, 0], 1.0, L, dtype=np.float64)
    q = keytree.quantise(p, [0, 0, 0], 1.0, L, dtype=np.float64)
    keys = []
    for x, y, z in zip(*[c.tolist() for c in q]):
        m = 0
        for k in range(L):
            m |= ((x >> k) & 1) << (3 * k + 2) | ((y >> k) & 1) << (3 * k + 1) | ((z >> k) & 1) << (3 * k)
        st, key, b = 0, 0, L
        while b >= 2:                              # two levels per lookup, as the kernel does
            e = int(tab[st * 64 + ((m >> (3 * (b - 2))) & 63)])
            key, st, b = key << 6 | (e & 63), e >> 6, b - 2
        if b:
            e = int(tab[1536 + st * 8 + (m & 7)])
            key = key << 3 | (e & 7)
        keys.append(key)
    assert np.array_equal(np.array(keys, dtype=np.uint64), ref)


def test_every_state_is_a_permutation_and_reachable():
    from paper_1506_04553_b200 import binding

    tab = binding.hilbert_state_tables()[1536:].reshape(24, 8)
    for s in range(24):
        assert sorted((tab[s] & 7).tolist()) == list(range(8))
    assert set((tab >> 3).ravel().tolist()) == set(range(24))
