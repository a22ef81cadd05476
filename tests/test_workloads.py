"""The seeded generators: shapes, structure and determinism of the five BASELINE.json configs."""
import numpy as np
import pytest

import workloads as W


def _distinct_within_constraints(inst):
    v = np.abs(inst.lits)
    for c in range(min(inst.m, 3000)):
        row = v[inst.row_ptr[c]:inst.row_ptr[c + 1]]
        assert np.unique(row).size == row.size


def test_config0_shape():
    c = W.config(0)
    assert (c.n, c.m, c.nnz, c.B, c.steps) == (50, 213, 639, 64, 200) and c.lr == 0.1
    assert c.X0.dtype == np.float32 and c.X0.shape == (64, 50) and np.abs(c.X0).max() <= 1
    assert c.plant is None and c.mask is None and np.all(c.types == W.AFS_OR)
    _distinct_within_constraints(c)


def test_config1_shape_and_plant():
    c = W.config(1)
    assert (c.n, c.m, c.B, c.steps) == (1000, 3450, 1024, 500)
    counts = np.bincount(c.types, minlength=7)
    assert list(counts) == [3000, 200, 100, 100, 0, 0, 50]
    L = c.lengths()
    for ty, lo, hi in [(W.AFS_OR, 3, 5), (W.AFS_XOR, 3, 8), (W.AFS_EO, 5, 20), (W.AFS_AMO, 5, 20), (W.AFS_CARD, 10, 40)]:
        sel = L[c.types == ty]
        assert sel.min() >= lo and sel.max() <= hi
    assert W.plant_satisfies(c, c.plant).all()
    kc, Lc = c.k[c.types == W.AFS_CARD], L[c.types == W.AFS_CARD]
    assert np.all(kc >= 1) and np.all(kc <= Lc - 1)
    _distinct_within_constraints(c)


def test_config2_duplicates():
    c = W.config(2)
    assert (c.n, c.m, c.nnz, c.B, c.steps) == (2000, 3600, 10800, 4096, 1000)
    assert np.all(c.lits > 0) and np.all(c.types == W.AFS_XOR)
    assert np.array_equal(c.lits[:5400], c.lits[5400:]) and np.array_equal(c.k[:1800], c.k[1800:])
    assert W.plant_satisfies(c, c.plant).all()


def test_config3_shape():
    c = W.config(3, B=32)
    assert (c.n, c.m, c.nnz, c.B, c.steps) == (100_000, 420_000, 1_260_000, 32, 300)
    assert W.plant_satisfies(c, c.plant).all()
    deg = np.bincount(np.abs(c.lits) - 1, minlength=c.n)
    assert 12.0 < deg.mean() < 13.2 and deg.max() < 45


def test_config4_shape_mask_and_thresholds():
    c = W.config(4, B=16)
    assert (c.n, c.m, c.steps) == (5000, 20500, 500)
    L = c.lengths()
    long = L > 3
    assert long.sum() == 500 and L[long].min() >= 256 and L[long].max() <= 1024
    assert list(np.bincount(c.types, minlength=7)) == [20000, 0, 0, 0, 100, 0, 400]
    assert W.plant_satisfies(c, c.plant).all()
    assert np.array_equal(W.true_counts(c, c.plant)[long], c.k[long])           # k := plant's true count (G22)
    assert (c.mask != 0).sum() == 2500 and np.array_equal(c.mask[c.mask != 0], c.plant[c.mask != 0])


def test_determinism_and_prefix_property():
    a, b = W.config(1), W.config(1)
    assert a.sha256() == b.sha256()
    small = W.config(1, B=64)
    assert np.array_equal(small.X0, a.X0[:64]) and np.array_equal(small.lits, a.lits)
    assert W.config(0).sha256() != W.config(0 + 0, B=32).sha256()


def test_tiny_mixed_covers_all_types():
    t = W.tiny_mixed(1, n=10)
    assert set(t.types.tolist()) == set(range(7))
    _distinct_within_constraints(t)
