"""Input generators: determinism, sub-range reproducibility, distribution sanity."""
import numpy as np

import workloads as w


def test_counter_based_and_deterministic():
    a = w.normal_field(123, 1000)
    b = w.normal_field(123, 400, start=300)
    assert np.array_equal(a[300:700], b)
    assert not np.array_equal(a, w.normal_field(124, 1000))
    big = w.normal_field(7, 200000)
    assert abs(big.mean()) < 0.01 and abs(big.std() - 1.0) < 0.01


def test_unit_vectors_and_configs():
    for i in (1, 2):
        c = w.get_config(i)
        m = c.initial_m()
        assert m.shape == c.n + (3,) and m.dtype == np.float64
        assert np.allclose(np.linalg.norm(m, axis=-1), 1.0, atol=1e-15)
    m2 = w.get_config(2).initial_m()
    assert abs(m2[..., 0].mean() - 1 / np.sqrt(1.01)) < 1e-3
    s = w.box_filter_renormalise(w.random_unit_vectors(3, (8, 8, 8)))
    assert np.allclose(np.linalg.norm(s, axis=-1), 1.0, atol=1e-15)
    r = w.random_unit_vectors(3, (8, 8, 8))
    # smoothing raises nearest-neighbour alignment
    assert np.mean(np.sum(s[1:] * s[:-1], -1)) > np.mean(np.sum(r[1:] * r[:-1], -1)) + 0.3


def test_sparse_sources_and_samples():
    m, ids = w.sparse_sources(5, (16, 8, 4), 6)
    assert 0 in ids and 16 * 8 * 4 - 1 in ids
    nz = np.flatnonzero(np.linalg.norm(m.reshape(-1, 3), axis=-1))
    assert np.array_equal(nz, ids)
    cells = w.sample_cells(1, (16, 8, 4), 50)
    assert cells.min() == 0 and cells.max() == 16 * 8 * 4 - 1 and len(np.unique(cells)) == len(cells)
