"""Seeded matrix coefficients with the structure of the paper's discretisation.

PAPER.md:34 (§1): row i of the implicit-Euler system is
    (sigma_i c_m,i / dt + sum_j a_ij) V_i - sum_j a_ij V_j = rhs_i,   a_ij = a_ji > 0
so the matrix is symmetric and strictly diagonally dominant.
BASELINE.json fixes the distributions:  a_ij ~ U[0.5, 2],  sigma c_m/dt ~ U[1, 10],
d_i = sigma c_m/dt + sum_j a_ij,  u_i = -a_{i,p(i)},  b ~ U[-1, 1].

This is input construction only (sums of positive numbers); no elimination,
substitution or any other step of the solver lives here.
"""
from __future__ import annotations

import numpy as np

from . import rng
from .morphology import Morphology


def global_parent(m: Morphology) -> np.ndarray:
    """int64 [N] global parent index (-1 at roots)."""
    sizes = np.diff(m.cell_offsets)
    gp = m.parent.astype(np.int64)
    gp += np.repeat(m.cell_offsets[:-1], sizes)
    gp[m.cell_offsets[:-1]] = -1
    return gp


def coefficients(m: Morphology, seed: int = rng.BASE_SEED, index_base: int = 0):
    """Return (d, u, sigma) as float64 arrays of length N.

    ``a`` and ``sigma`` are keyed by the global compartment index (+ index_base).
    d_i = (sigma_i + a_i) + (sum of a_c over children c, ascending c); roots have no a_i.
    u_i = -a_i, u_root = 0.
    """
    n = m.n
    idx = np.arange(n, dtype=np.uint64) + np.uint64(index_base)
    a = rng.uniform(seed, rng.STREAM_A, idx, 0.5, 2.0)
    a[m.cell_offsets[:-1]] = 0.0
    sigma = rng.uniform(seed, rng.STREAM_SIGMA, idx, 1.0, 10.0)
    del idx
    gp = global_parent(m)
    gp[m.cell_offsets[:-1]] = 0            # weight there is 0.0 anyway
    child_sum = np.bincount(gp, weights=a, minlength=n)
    del gp
    d = sigma + a
    d += child_sum
    u = -a
    u[m.cell_offsets[:-1]] = 0.0
    return d, u, sigma


def rhs(m: Morphology, seed: int = rng.BASE_SEED, step: int = 0, index_base: int = 0) -> np.ndarray:
    """b ~ U[-1, 1], keyed by (step, global compartment index): a fresh right-hand side
    per time step (config 4 uses step = 0..999)."""
    idx = np.arange(m.n, dtype=np.uint64) + np.uint64(index_base) + (np.uint64(step) << np.uint64(40))
    return rng.uniform(seed, rng.STREAM_B, idx, -1.0, 1.0)


def system(m: Morphology, seed: int = rng.BASE_SEED, dtype=np.float64, step: int = 0):
    """(d, u, b) for morphology m; fp32: generated in fp64 and rounded once."""
    d, u, _ = coefficients(m, seed)
    b = rhs(m, seed, step)
    if np.dtype(dtype) != np.float64:
        d, u, b = d.astype(dtype), u.astype(dtype), b.astype(dtype)
    return d, u, b
