"""Test-side helpers: dense assembly and tiny seeded systems.  Written in the tests on
purpose (not in oracle/): the pins must not be the oracle re-calling itself."""
from __future__ import annotations

import itertools

import numpy as np

import morphgen as mg


def dense_from_hines(p, d, u):
    """A[i,i] = d[i]; A[i,p[i]] = A[p[i],i] = u[i]."""
    n = len(d)
    A = np.zeros((n, n))
    A[np.arange(n), np.arange(n)] = d
    for i in range(1, n):
        A[i, p[i]] = u[i]
        A[p[i], i] = u[i]
    return A


def all_parent_arrays(n):
    """Every parent array with p[0] = -1 and 0 <= p[i] < i: (n-1)! trees."""
    for tail in itertools.product(*[range(i) for i in range(1, n)]):
        yield np.array((-1,) + tail, dtype=np.int32)


def random_parent(n, seed, chain_bias=0.6):
    """Random tree with p[i] < i; with probability chain_bias p[i] = i-1 (long branches)."""
    r = mg.rng.uniform01(seed, 77, np.arange(2 * n, dtype=np.uint64))
    p = np.empty(n, np.int32); p[0] = -1
    for i in range(1, n):
        p[i] = i - 1 if r[2 * i] < chain_bias else int(r[2 * i + 1] * i)
    return p


def system_for(p, seed=1, cell_offsets=None):
    """Seeded SDD coefficients (BASELINE.json distributions) for one or more cells."""
    p = np.asarray(p, np.int32)
    offs = np.array([0, len(p)], np.int64) if cell_offsets is None else np.asarray(cell_offsets, np.int64)
    m = mg.Morphology(p, offs)
    d, u, b = mg.system(m, seed)
    return m, d, u, b


def dfs_renumber(p):
    """Another valid numbering of the same tree (depth-first preorder).  Returns (perm, p_new)
    with perm[new] = old."""
    n = len(p)
    kids = [[] for _ in range(n)]
    for i in range(1, n):
        kids[p[i]].append(i)
    order, stack = [], [0]
    while stack:
        v = stack.pop()
        order.append(v)
        stack.extend(reversed(kids[v]))
    perm = np.array(order)
    inv = np.empty(n, np.int64); inv[perm] = np.arange(n)
    p_new = np.array([-1] + [inv[p[perm[k]]] for k in range(1, n)], np.int32)
    return perm, p_new


def rooted_at(parent, offs, pick):
    """The same cells (same undirected trees) rooted elsewhere: cell c is re-rooted at its compartment pick(c, n) and
    renumbered in breadth-first order from there, so that parent[i] < i holds again.  Returns (parent', perm, usrc) with
    perm[new] = old (global) and usrc[new] = the old compartment holding the coupling of new's edge to its parent --
    test-side construction of badly rooted inputs for the re-rooting pass (f2); shares nothing with oracle/ or the library."""
    parent = np.asarray(parent, np.int32); offs = np.asarray(offs, np.int64)
    newp = np.empty_like(parent); perm = np.empty(len(parent), np.int64); usrc = np.empty(len(parent), np.int64)
    for c in range(len(offs) - 1):
        lo, hi = int(offs[c]), int(offs[c + 1])
        n = hi - lo
        adj = [[] for _ in range(n)]
        for i in range(1, n):
            adj[i].append(int(parent[lo + i])); adj[int(parent[lo + i])].append(i)
        r = int(pick(c, n))
        order, par_old, seen = [r], {r: -1}, {r}
        for v in order:
            for w in sorted(adj[v]):
                if w not in seen:
                    seen.add(w); par_old[w] = v; order.append(w)
        new_of = {v: k for k, v in enumerate(order)}
        for k, v in enumerate(order):
            q = par_old[v]
            perm[lo + k] = lo + v
            newp[lo + k] = -1 if q < 0 else new_of[q]
            usrc[lo + k] = lo + (v if q < 0 or parent[lo + v] == q else q)
    return newp, perm, usrc
