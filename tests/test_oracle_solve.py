"""Pins for oracle/hines_oracle.c (CPU only).  Each pin is something other than the oracle:
LAPACK dense solves, scipy's banded solver, closed forms, exact rational fixtures, residuals
and invariants the paper's matrix properties imply.  A dropped term, wrong sign,
wrong index (e.g. the printed u[p[i]] of Listing 2) or transposed operand fails at least one."""
import json
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.linalg

import morphgen as mg
import oracle
from helpers import all_parent_arrays, dense_from_hines, dfs_renumber, random_parent, system_for

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _solve1(p, d, u, b):
    return oracle.hines_solve(p, np.array([0, len(p)]), d, u, b)


# ---- exact rational fixtures ------------------------------------------------------------
def test_exact_small_systems():
    cases = json.load(open(os.path.join(GOLDEN, "exact_small_systems.json")))["cases"]
    assert len(cases) >= 4
    for c in cases:
        p, d, u, b = c["p"], c["d"], c["u"], c["b"]
        xs = [Fraction(a, q) for a, q in zip(c["x_num"], c["x_den"])]
        n = len(p)
        # the fixture itself is checked exactly: A x = b in rationals
        for i in range(n):
            row = Fraction(d[i]) * xs[i]
            if i > 0:
                row += Fraction(u[i]) * xs[p[i]]
            for j in range(1, n):
                if p[j] == i:
                    row += Fraction(u[j]) * xs[j]
            assert row == Fraction(b[i]), (c["name"], i)
        x = _solve1(np.array(p, np.int32), np.array(d, float), np.array(u, float), np.array(b, float))
        np.testing.assert_allclose(x, [float(v) for v in xs], rtol=4e-16, atol=0)


# ---- dense Gaussian elimination (LAPACK) on every tree with n <= 7 ------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7])
def test_all_trees_vs_dense(n):
    count = 0
    for k, p in enumerate(all_parent_arrays(n)):
        _, d, u, b = system_for(p, seed=1000 + k)
        x = _solve1(p, d, u, b)
        xr = np.linalg.solve(dense_from_hines(p, d, u), b)
        np.testing.assert_allclose(x, xr, rtol=0, atol=5e-15 * max(1.0, np.abs(xr).max()))
        count += 1
    assert count == int(np.prod(np.arange(1, n)))   # (n-1)!


def test_printed_listing2_is_wrong():
    """Reading G1: Listing 2 as printed (u[p[i]] in the backward sweep)
    does not solve the system; the oracle's u[i] reading does.  Shows the dense pin is
    sensitive to exactly this index mistake."""
    p = np.array([-1, 0, 1, 1, 2, 2], np.int32)
    _, d, u, b = system_for(p, seed=5)
    xr = np.linalg.solve(dense_from_hines(p, d, u), b)
    dw, x = d.copy(), b.copy()
    for i in range(len(p) - 1, 0, -1):
        f = u[p[i]] / dw[i]
        dw[p[i]] -= f * u[p[i]]
        x[p[i]] -= f * x[i]
    x[0] /= dw[0]
    for i in range(1, len(p)):
        x[i] = (x[i] - u[i] * x[p[i]]) / dw[i]
    assert np.abs(x - xr).max() > 1e-3
    assert np.abs(_solve1(p, d, u, b) - xr).max() < 1e-14


@pytest.mark.parametrize("n,seed", [(12, 1), (50, 2), (200, 3), (200, 4)])
def test_random_trees_vs_dense(n, seed):
    p = random_parent(n, seed, chain_bias=0.5 if seed % 2 else 0.8)
    _, d, u, b = system_for(p, seed=seed)
    xr = np.linalg.solve(dense_from_hines(p, d, u), b)
    np.testing.assert_allclose(_solve1(p, d, u, b), xr, rtol=0, atol=2e-14)


def test_batch_cells_independent_vs_dense():
    """Several cells concatenated (reading S3): each block solved on its own."""
    ps = [random_parent(n, 10 + n) for n in (1, 2, 9, 30, 1, 17)]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    m, d, u, b = system_for(np.concatenate(ps), seed=9, cell_offsets=offs)
    x = oracle.hines_solve(m.parent, offs, d, u, b)
    for c, p in enumerate(ps):
        s = slice(offs[c], offs[c + 1])
        xr = np.linalg.solve(dense_from_hines(p, d[s], u[s]), b[s])
        np.testing.assert_allclose(x[s], xr, rtol=0, atol=2e-14)


# ---- cables: Thomas, banded library solver, Toeplitz closed form -------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 10, 1000])
def test_cable_vs_banded_and_thomas(n):
    p = np.arange(-1, n - 1, dtype=np.int32)
    _, d, u, b = system_for(p, seed=n)
    ab = np.zeros((3, n)); ab[1] = d; ab[0, 1:] = u[1:]; ab[2, :-1] = u[1:]
    xr = scipy.linalg.solve_banded((1, 1), ab, b)
    xh = _solve1(p, d, u, b)
    xt = oracle.thomas(d, u, b)
    np.testing.assert_allclose(xh, xr, rtol=0, atol=2e-15)
    # "If p[i] = i-1 holds, then Hines algorithm is equivalent to Thomas algorithm"
    assert np.array_equal(xh, xt)


def test_cable_toeplitz_closed_form():
    """Constant coefficients d = 2 cosh(theta), u = -1: the inverse is known in closed form,
    (T^-1)_{ij} = sinh(i th) sinh((n+1-j) th) / (sinh th sinh((n+1) th)),  i <= j (1-based)."""
    n, th = 40, 0.3
    p = np.arange(-1, n - 1, dtype=np.int32)
    d = np.full(n, 2 * np.cosh(th)); u = np.full(n, -1.0); u[0] = 0.0
    for j in (1, 7, 40):
        b = np.zeros(n); b[j - 1] = 1.0
        i = np.arange(1, n + 1)
        lo, hi = np.minimum(i, j), np.maximum(i, j)
        xr = np.sinh(lo * th) * np.sinh((n + 1 - hi) * th) / (np.sinh(th) * np.sinh((n + 1) * th))
        np.testing.assert_allclose(_solve1(p, d, u, b), xr, rtol=1e-12, atol=0)
        np.testing.assert_allclose(oracle.thomas(d, u, b), xr, rtol=1e-12, atol=0)


# ---- star tree: pins the hand-off at a branch point and the sibling sum -------------------
@pytest.mark.parametrize("k", [1, 2, 5, 33])
def test_star_closed_form(k):
    p = np.array([-1] + [0] * k, np.int32)
    _, d, u, b = system_for(p, seed=k)
    x0 = (b[0] - np.sum(u[1:] * b[1:] / d[1:])) / (d[0] - np.sum(u[1:] ** 2 / d[1:]))
    xr = np.concatenate([[x0], (b[1:] - u[1:] * x0) / d[1:]])
    np.testing.assert_allclose(_solve1(p, d, u, b), xr, rtol=1e-14, atol=0)


def test_single_compartment_and_unused_root_u():
    """S16: n = 1 gives x = b/d.  S2: u[root] can never reach the result (NaN poison)."""
    x = _solve1(np.array([-1], np.int32), np.array([4.0]), np.array([np.nan]), np.array([2.0]))
    assert x[0] == 0.5
    p = random_parent(25, 3)
    _, d, u, b = system_for(p, seed=3)
    u2 = u.copy(); u2[0] = np.nan
    assert np.array_equal(_solve1(p, d, u, b), _solve1(p, d, u2, b))


# ---- properties at any size ------------------------------------------------------------------
@pytest.fixture(scope="module", params=[0, 1, 2, 3, 4])
def cfg_system(request):
    scale = {0: 1.0, 1: 0.02, 2: 0.02, 3: 0.005, 4: 1.0}[request.param]
    m = mg.make_config(request.param, scale)
    d, u, sigma = mg.coefficients(m)
    b = mg.rhs(m)
    return m, d, u, b, sigma


def test_generator_structure(cfg_system):
    """symmetric (one u per edge), strictly diagonally dominant; p[i] < i."""
    m, d, u, b, sigma = cfg_system
    gp = mg.global_parent(m)
    assert (gp < np.arange(m.n)).all() and (gp[m.cell_offsets[:-1]] == -1).all()
    offdiag = np.abs(u) + np.bincount(np.maximum(gp, 0), weights=np.where(gp >= 0, np.abs(u), 0.0), minlength=m.n)
    assert (d > offdiag).all()
    assert (u[gp >= 0] <= -0.5).all() and (u[gp >= 0] >= -2.0).all() and (u[gp < 0] == 0).all()
    assert (sigma >= 1).all() and (sigma < 10).all() and (np.abs(b) <= 1).all()


def test_residual(cfg_system):
    m, d, u, b, _ = cfg_system
    x = oracle.hines_solve(m.parent, m.cell_offsets, d, u, b)
    # residual recomputed here from (d,u,p) with numpy, not with the oracle's matvec
    gp = mg.global_parent(m)
    nz = gp >= 0
    y = d * x
    y[nz] += u[nz] * x[gp[nz]]
    y += np.bincount(gp[nz], weights=u[nz] * x[nz], minlength=m.n)
    r = np.abs(y - b)
    cell = np.repeat(np.arange(m.ncells), np.diff(m.cell_offsets))
    rmax = np.zeros(m.ncells); np.maximum.at(rmax, cell, r)
    bmax = np.zeros(m.ncells); np.maximum.at(bmax, cell, np.abs(b))
    assert (rmax / bmax).max() < 1e-12
    # and the oracle's own residual helper agrees with that number
    np.testing.assert_allclose(oracle.residual(m.parent, m.cell_offsets, d, u, b, x), rmax / bmax,
                               rtol=0, atol=1e-15)


def test_row_sums_give_ones(cfg_system):
    """b := A 1 (row sums accumulated in floating point from d, u, p)  =>  x = 1."""
    m, d, u, _, _ = cfg_system
    gp = mg.global_parent(m)
    nz = gp >= 0
    b1 = d.copy()
    b1[nz] += u[nz]
    b1 += np.bincount(gp[nz], weights=u[nz], minlength=m.n)
    x = oracle.hines_solve(m.parent, m.cell_offsets, d, u, b1)
    assert np.abs(x - 1.0).max() < 5e-15


def test_pivot_and_multiplier_invariants(cfg_system):
    """I1: d'[i] >= sigma_i + a_{i,p(i)} > 0; I2: |f| = |u/d'| < 1 (no pivoting)."""
    m, d, u, _, sigma = cfg_system
    dw = oracle.pivots(m.parent, m.cell_offsets, d, u)
    assert (dw - (sigma + np.abs(u)) >= -1e-12).all()
    assert (np.abs(u) / dw < 1.0).all()


def test_maximum_principle(cfg_system):
    """I3: A is an M-matrix with A 1 = sigma  =>  ||x||_inf <= ||b||_inf / min sigma, b>=0 => x>=0."""
    m, d, u, b, sigma = cfg_system
    x = oracle.hines_solve(m.parent, m.cell_offsets, d, u, b)
    assert np.abs(x).max() <= np.abs(b).max() / sigma.min() + 1e-15
    xp = oracle.hines_solve(m.parent, m.cell_offsets, d, u, np.abs(b))
    assert (xp >= 0).all()


def test_linearity_and_renumbering():
    p = random_parent(120, 8, chain_bias=0.7)
    m, d, u, b = system_for(p, seed=8)
    b2 = mg.rhs(m, step=1)
    x1, x2 = _solve1(p, d, u, b), _solve1(p, d, u, b2)
    x12 = _solve1(p, d, u, 2.0 * b - 3.0 * b2)
    np.testing.assert_allclose(x12, 2.0 * x1 - 3.0 * x2, rtol=0, atol=1e-14)
    # another valid numbering (depth-first) of the same tree gives the same solution
    perm, p_new = dfs_renumber(p)
    x_new = _solve1(p_new, d[perm], np.where(np.arange(len(p)) == 0, 0.0, u[perm]), b[perm])
    np.testing.assert_allclose(x_new, x1[perm], rtol=0, atol=1e-14)


# ---- the parity metric itself (reading S15) and the range entry: pinned against numpy, not against themselves ----
def _rel_err_numpy(offs, xa, xb):
    out = np.empty(len(offs) - 1)
    for c in range(len(offs) - 1):
        a, b_ = xa[offs[c]:offs[c + 1]], xb[offs[c]:offs[c + 1]]
        diff = np.abs(a - b_)
        e = np.nan if np.isnan(diff).any() else diff.max()
        nrm = np.abs(b_).max()
        out[c] = e / nrm if nrm > 0 else e
    return out


def test_rel_err_matches_numpy_per_cell():
    offs = np.array([0, 3, 4, 10, 210, 211], np.int64)
    r = mg.rng.uniform(5, 91, np.arange(2 * offs[-1], dtype=np.uint64), -2.0, 2.0)
    xb = r[:offs[-1]].copy()
    xa = xb + 1e-9 * r[offs[-1]:]
    err = oracle.rel_err(offs, xa, xb)
    np.testing.assert_allclose(err, _rel_err_numpy(offs, xa, xb), rtol=1e-15, atol=0)
    assert err.shape == (5,) and (err > 0).all()
    # the value is the per-cell ratio, not a global one: scaling one cell's reference scales only that cell's error
    xb2, xa2 = xb.copy(), xa.copy()
    xb2[3:4] *= 1e6; xa2[3:4] = xb2[3:4] + (xa[3:4] - xb[3:4])
    err2 = oracle.rel_err(offs, xa2, xb2)
    assert err2[1] == pytest.approx(err[1] * 1e-6, rel=1e-6) and np.array_equal(np.delete(err2, 1), np.delete(err, 1))


@pytest.mark.parametrize("pos", ["first", "middle", "last"])
def test_rel_err_nan_is_sticky_and_local(pos):
    """A NaN at any position of a cell gives NaN for that cell and only for that cell (the round-1 checker
    let a later finite element overwrite it)."""
    offs = np.array([0, 3, 8, 11], np.int64)
    xb = np.array([1, 2, 4, 0.5, 2, 3, 1, 1, 7, 8, 9], np.float64)
    xa = xb + 1e-3
    k = {"first": 3, "middle": 5, "last": 7}[pos]
    xa[k] = np.nan
    err = oracle.rel_err(offs, xa, xb)
    assert np.isnan(err[1]) and np.isfinite(err[0]) and np.isfinite(err[2])
    np.testing.assert_allclose(err[[0, 2]], [1e-3 / 4, 1e-3 / 9], rtol=1e-12)
    # the probe of VERDICT.md round 1: an isolated NaN followed by finite elements
    e2 = oracle.rel_err(np.array([0, 3, 5], np.int64), np.array([1, np.nan, 3, 0, 0.0]), np.array([1, 2, 4, 0, 1e-3]))
    assert np.isnan(e2[0]) and e2[1] == 1.0
    # NaN in the reference is not hidden either
    e3 = oracle.rel_err(np.array([0, 2], np.int64), np.array([1.0, 2.0]), np.array([np.nan, 2.0]))
    assert np.isnan(e3[0])


def test_rel_err_zero_reference_is_absolute():
    offs = np.array([0, 2, 4], np.int64)
    err = oracle.rel_err(offs, np.array([1e-3, -2e-3, 1.0, 1.0]), np.array([0.0, 0.0, 1.0, 1.0]))
    assert err[0] == 2e-3 and err[1] == 0.0


def test_solve_range_equals_dense_and_full_solve():
    """hines_solve_range over any split of the cells: bit-equal to hines_solve, and each range on its own equal to
    dense solves of its cells; cells outside the range are not touched."""
    ps = [random_parent(n, 30 + n, 0.6) for n in (1, 17, 40, 5, 64, 2, 33)]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])]).astype(np.int64)
    m, d, u, b = system_for(np.concatenate(ps), seed=21, cell_offsets=offs)
    x_full = oracle.hines_solve(m.parent, offs, d, u, b)
    par = np.ascontiguousarray(m.parent, np.int32)
    for cuts in ([0, 7], [0, 3, 7], [0, 1, 2, 6, 7], [0, 5, 5, 7]):
        x = np.full(m.n, -77.0); dw = np.empty(m.n)
        for c0, c1 in zip(cuts[:-1], cuts[1:]):
            before = x.copy()
            oracle.hines_solve_range(c0, c1, par, offs, d, u, b, x, dw)
            untouched = np.ones(m.n, bool); untouched[offs[c0]:offs[c1]] = False
            assert np.array_equal(x[untouched], before[untouched])
        assert np.array_equal(x, x_full)
    for c in range(len(ps)):
        A = dense_from_hines(ps[c], d[offs[c]:offs[c + 1]], u[offs[c]:offs[c + 1]])
        np.testing.assert_allclose(x_full[offs[c]:offs[c + 1]], np.linalg.solve(A, b[offs[c]:offs[c + 1]]), rtol=0, atol=2e-15)


def test_pivots_equal_schur_complements():
    """oracle_pivots: d'[i] is the Schur complement of the sub-tree below i onto i, i.e. 1 / [A_sub^-1]_{ii} for
    the principal sub-matrix of i and its descendants (dense inverse), not only the inequalities I1/I2."""
    p = random_parent(40, 3, 0.5)
    m, d, u, _ = system_for(p, seed=4)
    dw = oracle.pivots(m.parent, m.cell_offsets, d, u)
    A = dense_from_hines(p, d, u)
    n = len(p)
    desc = [[i] for i in range(n)]
    for i in range(n - 1, 0, -1):
        desc[p[i]] += desc[i]
    for i in range(n):
        idx = sorted(desc[i])
        S = np.linalg.inv(A[np.ix_(idx, idx)])
        assert dw[i] == pytest.approx(1.0 / S[idx.index(i), idx.index(i)], rel=1e-13)


# ---- f3: factor once / solve many ----------------------------------------------
def test_factor_then_rhs_is_bit_equal_to_the_full_solve_and_to_dense():
    ps = [random_parent(n, 50 + n, 0.6) for n in (1, 2, 30, 200, 9)]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])]).astype(np.int64)
    m, d, u, b = system_for(np.concatenate(ps), seed=31, cell_offsets=offs)
    dw, f = oracle.hines_factor(m.parent, offs, d, u)
    assert np.array_equal(dw, oracle.pivots(m.parent, offs, d, u))
    for step in range(3):                                    # the same factors, a fresh right-hand side per step
        bs = mg.rhs(m, step=step)
        x = oracle.hines_solve_rhs(m.parent, offs, dw, f, u, bs)
        assert np.array_equal(x, oracle.hines_solve(m.parent, offs, d, u, bs))
        for c in range(len(ps)):
            A = dense_from_hines(ps[c], d[offs[c]:offs[c + 1]], u[offs[c]:offs[c + 1]])
            np.testing.assert_allclose(x[offs[c]:offs[c + 1]], np.linalg.solve(A, bs[offs[c]:offs[c + 1]]), rtol=0, atol=2e-15)
    # the multipliers: f[i] = A[i,p] / d'[i]; L D L^T with L = I + (f placed at (p[i], i)) reproduces A
    c = 3
    p = ps[c]; sl = slice(offs[c], offs[c + 1])
    n = len(p)
    Lm = np.eye(n)
    for i in range(1, n):
        Lm[p[i], i] = f[sl][i]
    np.testing.assert_allclose(Lm @ np.diag(dw[sl]) @ Lm.T, dense_from_hines(p, d[sl], u[sl]), rtol=0, atol=1e-13)
