"""The seeded input generators (inputs/): same bits from every implementation."""
import numpy as np
import torch

from inputs import CONFIGS, g_uniform, ring_bonds, sample_indices, start_vector_np, start_vector_torch, torus_bonds
from inputs.vectors import _g_scalar


def test_counter_generator_scalar_vs_numpy():
    idx = np.array([0, 1, 2, 12345, 2**31 - 1, 2**31, 2**32 + 7, 2363904399], dtype=np.int64)
    v = g_uniform(12043429, idx)
    for j, x in zip(idx, v):
        assert x == _g_scalar(12043429, int(j))
    assert np.all(v >= -1.0) and np.all(v < 1.0)


def test_counter_generator_torch_matches_numpy():
    for seed in (1, 12043425, 2**63 + 5):
        a = start_vector_np(seed, 100003, chunk=4096)
        b = start_vector_torch(seed, 100003, "cpu", chunk=7001).numpy()
        assert np.array_equal(a, b)
    # element access at large offsets equals the scalar definition
    big = np.array([2**31 + 11, 2363904399], dtype=np.int64)
    assert np.array_equal(g_uniform(7, big), [_g_scalar(7, int(j)) for j in big])


def test_generator_statistics():
    v = start_vector_np(3, 1 << 18)
    assert abs(v.mean()) < 5e-3 and abs(v.var() - 1.0 / 3.0) < 5e-3


def test_lattices():
    assert ring_bonds(4) == [(0, 1), (1, 2), (2, 3), (3, 0)]
    tb = torus_bonds(4, 4)
    assert len(tb) == 32 and len({(min(a, b), max(a, b)) for a, b in tb}) == 32
    deg = np.zeros(16, int)
    for a, b in tb:
        deg[a] += 1
        deg[b] += 1
    assert np.all(deg == 4)


def test_configs_dims():
    assert CONFIGS["C1"].dim == 4900
    assert CONFIGS["C2"].dim == 853776
    assert CONFIGS["C3"].dim == 4368 ** 2
    assert CONFIGS["C4"].dim == 12870 ** 2
    assert CONFIGS["C5"].dim == 48620 ** 2 == 2363904400


def test_sample_indices():
    s = sample_indices(5, 1000, 50)
    assert s[0] == 0 and s[-1] == 999 and np.all(np.diff(s) > 0)
    assert np.array_equal(s, sample_indices(5, 1000, 50))
