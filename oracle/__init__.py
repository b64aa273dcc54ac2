"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of the plain-C oracle (hines_oracle.c: PAPER.md Listings 1-2;
tables_oracle.c: PAPER.md:108-138 tables).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It imports nothing
from paper_1810_12742_b200 and shares no code with it.

Parity pins: every function below is pinned by tests/test_oracle_*.py against something
other than itself (dense LAPACK solves incl. all trees with n <= 7, banded solver, closed
forms, residual, x = 1 identity, brute-force tables).  The only unpinned items are the
*policy* tables (work items / lanes), which the paper does not fix: see DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_tables_count.restype = C.c_int64
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _prep(parent, cell_offsets):
    parent = np.ascontiguousarray(parent, dtype=np.int32)
    offs = np.ascontiguousarray(cell_offsets, dtype=np.int64)
    return parent, offs, C.c_int64(len(offs) - 1)


def hines_solve(parent, cell_offsets, d, u, b):
    """x = A^-1 b per cell by Listing 2 (reading G1), fp64."""
    parent, offs, nc = _prep(parent, cell_offsets)
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64)
    b = np.ascontiguousarray(b, np.float64)
    x = np.empty_like(d); dw = np.empty_like(d)
    lib().oracle_hines_solve(nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(d, C.c_double),
                             _p(u, C.c_double), _p(b, C.c_double), _p(x, C.c_double), _p(dw, C.c_double))
    return x


def hines_solve_range(c0, c1, parent, cell_offsets, d, u, b, x, dw):
    """In-place variant on cells [c0, c1) (arrays preallocated, contiguous, right dtypes).
    The ctypes call releases the GIL, so a thread pool gives a plain parallel-for over cells."""
    lib().oracle_hines_solve_range(C.c_int64(c0), C.c_int64(c1), _p(cell_offsets, C.c_int64),
                                   _p(parent, C.c_int32), _p(d, C.c_double), _p(u, C.c_double),
                                   _p(b, C.c_double), _p(x, C.c_double), _p(dw, C.c_double))


def thomas(d, u, b):
    """Listing 1 (reading G2) on one tridiagonal system."""
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64)
    b = np.ascontiguousarray(b, np.float64)
    x = np.empty_like(d); dw = np.empty_like(d)
    lib().oracle_thomas(C.c_int64(len(d)), _p(d, C.c_double), _p(u, C.c_double), _p(b, C.c_double),
                        _p(x, C.c_double), _p(dw, C.c_double))
    return x


def matvec(parent, cell_offsets, d, u, x):
    parent, offs, nc = _prep(parent, cell_offsets)
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64)
    x = np.ascontiguousarray(x, np.float64); y = np.empty_like(d)
    lib().oracle_matvec(nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(d, C.c_double),
                        _p(u, C.c_double), _p(x, C.c_double), _p(y, C.c_double))
    return y


def residual(parent, cell_offsets, d, u, b, x):
    """per cell ||Ax-b||_inf / ||b||_inf."""
    parent, offs, nc = _prep(parent, cell_offsets)
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64)
    b = np.ascontiguousarray(b, np.float64); x = np.ascontiguousarray(x, np.float64)
    y = np.empty_like(d); res = np.empty(nc.value, np.float64)
    lib().oracle_residual(nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(d, C.c_double),
                          _p(u, C.c_double), _p(b, C.c_double), _p(x, C.c_double),
                          _p(y, C.c_double), _p(res, C.c_double))
    return res


def pivots(parent, cell_offsets, d, u):
    parent, offs, nc = _prep(parent, cell_offsets)
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64)
    dw = np.empty_like(d)
    lib().oracle_pivots(nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(d, C.c_double),
                        _p(u, C.c_double), _p(dw, C.c_double))
    return dw


def rel_err(cell_offsets, xa, xb):
    """per cell ||xa-xb||_inf / ||xb||_inf (reading S15); NaN in xa gives NaN."""
    offs = np.ascontiguousarray(cell_offsets, np.int64)
    xa = np.ascontiguousarray(xa, np.float64); xb = np.ascontiguousarray(xb, np.float64)
    err = np.empty(len(offs) - 1, np.float64)
    lib().oracle_rel_err(C.c_int64(len(offs) - 1), _p(offs, C.c_int64), _p(xa, C.c_double),
                         _p(xb, C.c_double), _p(err, C.c_double))
    return err


@dataclass
class Tables:
    cell_branch_offsets: np.ndarray
    branch_start: np.ndarray
    branch_len: np.ndarray
    branch_parent_comp: np.ndarray
    branch_parent_branch: np.ndarray
    branch_level: np.ndarray
    cell_nlevels: np.ndarray
    cell_level_offsets: np.ndarray
    level_count: np.ndarray
    level_list: np.ndarray
    child_offsets: np.ndarray
    child_ids: np.ndarray


def tables(parent, cell_offsets) -> Tables:
    """Canonical (policy-free) scheduler tables T1-T7 (readings S4, S5, S7)."""
    parent, offs, nc = _prep(parent, cell_offsets)
    ncells = nc.value
    nb = lib().oracle_tables_count(nc, _p(offs, C.c_int64), _p(parent, C.c_int32))
    if nb < 0:
        raise ValueError("malformed parent array")
    i32 = lambda n: np.empty(max(n, 0), np.int32)
    i64 = lambda n: np.empty(max(n, 0), np.int64)
    t = Tables(i64(ncells + 1), i32(nb), i32(nb), i32(nb), i32(nb), i32(nb), i32(ncells),
               i64(ncells + 1), i32(nb), i32(nb), i64(nb + 1), i32(nb - ncells))
    nlc = C.c_int64(0)
    rc = lib().oracle_tables_build(
        nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(t.cell_branch_offsets, C.c_int64),
        _p(t.branch_start, C.c_int32), _p(t.branch_len, C.c_int32), _p(t.branch_parent_comp, C.c_int32),
        _p(t.branch_parent_branch, C.c_int32), _p(t.branch_level, C.c_int32),
        _p(t.cell_nlevels, C.c_int32), _p(t.cell_level_offsets, C.c_int64),
        _p(t.level_count, C.c_int32), C.c_int64(nb), C.byref(nlc),
        _p(t.level_list, C.c_int32), _p(t.child_offsets, C.c_int64), _p(t.child_ids, C.c_int32))
    assert rc == 0
    t.level_count = t.level_count[:nlc.value].copy()
    return t


def level_mean_split(parent, cell_offsets):
    """f1, the paper's branch splitting (reading F1): per branch the piece lengths (from the top of
    the branch) and piece levels, plus the per-level {sum, count} statistics.  Returns (piece_offsets[nbranches+1],
    piece_len, piece_level, level_stat[2*nlevels]) with pieces grouped by global branch index."""
    t = tables(parent, cell_offsets)
    nb = len(t.branch_len)
    ncomp = int(np.asarray(cell_offsets)[-1])
    pb = np.empty(ncomp, np.int64); pl = np.empty(ncomp, np.int32); pv = np.empty(ncomp, np.int32)
    ls = np.empty(ncomp, np.int64); lc = np.empty(ncomp, np.int64)
    nlev = C.c_int64(0)
    lib().oracle_level_mean_split.restype = C.c_int64
    npieces = lib().oracle_level_mean_split(
        C.c_int64(len(t.cell_branch_offsets) - 1), _p(t.cell_branch_offsets, C.c_int64), _p(t.branch_len, C.c_int32),
        _p(t.branch_parent_branch, C.c_int32), _p(pb, C.c_int64), _p(pl, C.c_int32), _p(pv, C.c_int32),
        _p(ls, C.c_int64), _p(lc, C.c_int64), C.byref(nlev))
    assert npieces >= nb
    pb, pl, pv = pb[:npieces], pl[:npieces], pv[:npieces]
    order = np.argsort(pb, kind="stable")                 # by branch; inside a branch the emission order = top-down
    offs = np.concatenate([[0], np.cumsum(np.bincount(pb, minlength=nb))]).astype(np.int64)
    stat = np.empty(2 * nlev.value, np.int64)
    stat[0::2] = ls[:nlev.value]; stat[1::2] = lc[:nlev.value]
    return offs, pl[order].copy(), pv[order].copy(), stat


def reroot(parent, cell_offsets):
    """f2, tree re-rooting (readings R1-R3): per cell the compartment that minimises the depth of the
    tree becomes the root and the compartments are renumbered branch by branch, breadth first.  Returns a dict:
    root[ncells] (old cell-local index), depth_before / depth_after[ncells], perm[N] (GLOBAL: new -> old), new_parent[N]
    (cell-local), usrc[N] (GLOBAL old index whose u holds the coupling of the new compartment's edge to its parent)."""
    parent, offs, _ = _prep(parent, cell_offsets)
    nc, n = len(offs) - 1, int(offs[-1])
    root = np.empty(nc, np.int32); db = np.empty(nc, np.int32); da = np.empty(nc, np.int32)
    perm = np.empty(n, np.int64); newp = np.empty(n, np.int32); usrc = np.empty(n, np.int64)
    fn = lib().oracle_reroot_cell
    fn.restype = C.c_int32
    for c in range(nc):
        lo, hi = int(offs[c]), int(offs[c + 1])
        m = hi - lo
        pc = np.ascontiguousarray(parent[lo:hi], np.int32)
        pm = np.empty(m, np.int32); npar = np.empty(m, np.int32); us = np.empty(m, np.int32)
        r, d0 = C.c_int32(0), C.c_int32(0)
        dep = fn(C.c_int32(m), _p(pc, C.c_int32), C.byref(r), C.byref(d0), _p(pm, C.c_int32), _p(npar, C.c_int32), _p(us, C.c_int32))
        assert dep >= 0
        root[c], db[c], da[c] = r.value, d0.value, dep
        perm[lo:hi] = pm.astype(np.int64) + lo; newp[lo:hi] = npar; usrc[lo:hi] = us.astype(np.int64) + lo
    return dict(root=root, depth_before=db, depth_after=da, perm=perm, new_parent=newp, usrc=usrc)


def hines_factor(parent, cell_offsets, d, u):
    """f3: the part of Listing 2 that touches only d and u.  Returns (dw, f): pivots and multipliers."""
    parent, offs, nc = _prep(parent, cell_offsets)
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64)
    dw = np.empty_like(d); f = np.empty_like(d)
    lib().oracle_hines_factor(nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(d, C.c_double), _p(u, C.c_double),
                              _p(dw, C.c_double), _p(f, C.c_double))
    return dw, f


def hines_solve_rhs(parent, cell_offsets, dw, f, u, b):
    """f3: x = A^-1 b from the factors of hines_factor (the part of Listing 2 that touches b)."""
    parent, offs, nc = _prep(parent, cell_offsets)
    dw = np.ascontiguousarray(dw, np.float64); f = np.ascontiguousarray(f, np.float64)
    u = np.ascontiguousarray(u, np.float64); b = np.ascontiguousarray(b, np.float64)
    x = np.empty_like(b)
    lib().oracle_hines_solve_rhs(nc, _p(offs, C.c_int64), _p(parent, C.c_int32), _p(dw, C.c_double), _p(f, C.c_double),
                                 _p(u, C.c_double), _p(b, C.c_double), _p(x, C.c_double))
    return x
