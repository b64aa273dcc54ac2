"""The seeded input generators: determinism, ranges, and the BASELINE.json sizes."""
import numpy as np

import morphgen as mg
from morphgen import rng


def test_hash_matches_scalar_twin_and_is_order_free():
    idx = np.array([0, 1, 2, 12345678901, 2**40 + 17], dtype=np.uint64)
    h = rng.hash64(rng.BASE_SEED, rng.STREAM_A, idx)
    for i, v in zip(idx, h):
        assert int(v) == rng.hash64_scalar(rng.BASE_SEED, rng.STREAM_A, int(i))
    assert np.array_equal(rng.hash64(rng.BASE_SEED, rng.STREAM_A, idx[::-1]), h[::-1])
    assert not np.array_equal(rng.hash64(rng.BASE_SEED, rng.STREAM_B, idx), h)


def test_uniform_range_and_moments():
    r = rng.uniform01(1, 2, np.arange(200000, dtype=np.uint64))
    assert r.min() >= 0.0 and r.max() < 1.0
    assert abs(r.mean() - 0.5) < 5e-3 and abs(r.var() - 1 / 12) < 2e-3


def test_config_sizes_match_baseline():
    m0 = mg.make_config(0)
    assert m0.ncells == 64 and m0.n == 64 * 75
    m1 = mg.make_config(1, 0.01)
    assert m1.ncells == 100 and m1.n == 100_000
    m2 = mg.make_config(2, 0.1)
    per = np.diff(m2.cell_offsets)
    nbr = len(m2.gen_branch_len) / m2.ncells
    assert 3500 < per.mean() < 4600 and 170 < nbr < 230           # "~4,000 unknowns, ~200 branches"
    assert m2.gen_branch_len.min() >= 1 and m2.gen_branch_len.max() <= 40
    assert m2.gen_branch_level.max() == 12                          # "depth <= 12"
    m3 = mg.make_config(3, 0.02)
    per = np.diff(m3.cell_offsets); large = m3.meta["large"]
    assert 0.17 < large.mean() < 0.23
    assert 150 < per[~large].mean() < 260 and 8500 < per[large].mean() < 11500
    m4 = mg.make_config(4)
    assert m4.ncells == 1 and m4.n == 1_310_710 and len(m4.gen_branch_len) == 131_071


def test_cells_do_not_depend_on_batch_size():
    a = mg.make_config(2, 0.001)
    b = mg.make_config(2, 0.002)
    n = a.n
    assert np.array_equal(a.parent, b.parent[:n]) and np.array_equal(a.cell_offsets, b.cell_offsets[:a.ncells + 1])
    da, ua, _ = mg.coefficients(a); db, ub, _ = mg.coefficients(b)
    # d of the last compartment of `a` has no children outside `a`, so the prefix agrees exactly
    assert np.array_equal(da, db[:n]) and np.array_equal(ua, ub[:n])


def test_fresh_rhs_per_step():
    m = mg.make_config(0)
    b0, b1 = mg.rhs(m, step=0), mg.rhs(m, step=1)
    assert not np.array_equal(b0, b1) and np.array_equal(b0, mg.rhs(m, step=0))
    d32, u32, b32 = mg.system(m, dtype=np.float32)
    d64, _, _ = mg.system(m)
    assert d32.dtype == np.float32 and np.array_equal(d32, d64.astype(np.float32))
