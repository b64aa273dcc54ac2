"""Pins of the re-rooting oracle (oracle/reroot_oracle.c; readings R1-R3 of DESIGN.md) and, below
them, the library's hines_reroot against the oracle, bit for bit.  CPU only."""
import json
import os

import numpy as np
import pytest

import oracle
from helpers import random_parent

HERE = os.path.dirname(os.path.abspath(__file__))


def _depth(parent):
    d = np.zeros(len(parent), np.int64)
    for i in range(1, len(parent)):
        d[i] = d[parent[i]] + 1
    return int(d.max())


def _check_invariants(parent, offs, r):
    n = int(offs[-1])
    assert sorted(r["perm"].tolist()) == list(range(n))
    for c in range(len(offs) - 1):
        lo, hi = int(offs[c]), int(offs[c + 1])
        npar = r["new_parent"][lo:hi]
        assert npar[0] == -1 and all(0 <= npar[k] < k for k in range(1, hi - lo))
        assert r["perm"][lo] == lo + r["root"][c]
        assert ((r["perm"][lo:hi] >= lo) & (r["perm"][lo:hi] < hi)).all()
        assert _depth(npar) == r["depth_after"][c] and _depth(parent[lo:hi]) == r["depth_before"][c]
        # a branch of the new tree is a run of consecutive indices ("continuous indices"): a compartment
        # whose parent has exactly one child follows its parent directly
        nch = np.bincount(npar[1:], minlength=hi - lo)
        for k in range(1, hi - lo):
            if nch[npar[k]] == 1:
                assert npar[k] == k - 1
        # the same undirected edges, and usrc names the old child end of each
        old_edges = {(lo + i, lo + int(parent[lo + i])) for i in range(1, hi - lo)}
        for k in range(1, hi - lo):
            a, b = int(r["perm"][lo + k]), int(r["perm"][lo + npar[k]])
            assert ((a, b) in old_edges) != ((b, a) in old_edges)
            assert int(r["usrc"][lo + k]) == (a if (a, b) in old_edges else b)


def test_path_goes_to_its_middle():
    """Closed form: a path of n compartments rooted at one end has depth n - 1; its centre gives ceil((n - 1) / 2);
    of the two centres of an even path the larger index is taken (reading R2)."""
    for n in (1, 2, 3, 6, 7, 40, 41):
        parent = np.arange(-1, n - 1, dtype=np.int32)
        r = oracle.reroot(parent, [0, n])
        assert r["depth_before"][0] == n - 1 and r["depth_after"][0] == n // 2
        assert r["root"][0] == n // 2
        _check_invariants(parent, np.array([0, n]), r)


def test_star_and_leaf_rooted_star():
    """Closed form: a star rooted at a leaf (depth 2) is re-rooted at its hub (depth 1); rooted at the hub it stays."""
    n = 9
    hub_rooted = np.array([-1] + [0] * (n - 1), np.int32)
    leaf_rooted = np.array([-1, 0] + [1] * (n - 2), np.int32)
    r = oracle.reroot(hub_rooted, [0, n])
    assert r["root"][0] == 0 and r["depth_after"][0] == 1 and (r["perm"] == np.arange(n)).all()
    r = oracle.reroot(leaf_rooted, [0, n])
    assert r["root"][0] == 1 and r["depth_before"][0] == 2 and r["depth_after"][0] == 1
    _check_invariants(leaf_rooted, np.array([0, n]), r)


def test_paper_example_weak_pin():
    """"In the example, this would be the compartment with index 7."  Figure 1.1 is missing from the text;
    the tree inferred for it (five branches of five compartments, level widths 1-2-2; tests/golden/reroot_example.json)
    has the minimisers {6, 7} with depth 8 against 14 for root 0.  Weak pin: it fixes reading R2 (the larger index)."""
    g = json.load(open(os.path.join(HERE, "golden", "reroot_example.json")))
    parent = np.array(g["parent"], np.int32)
    r = oracle.reroot(parent, [0, len(parent)])
    assert r["root"][0] == g["root"] == 7
    assert r["depth_before"][0] == g["depth_root0"] and r["depth_after"][0] == g["depth_min"]
    _check_invariants(parent, np.array([0, len(parent)]), r)


def test_depth_is_half_the_diameter():
    """Textbook: the smallest eccentricity of a tree is ceil(diameter / 2); diameter by brute force here."""
    rng = np.random.default_rng(5)
    for trial in range(30):
        n = int(rng.integers(2, 60))
        parent = random_parent(n, 100 + trial, float(rng.uniform(0.2, 0.95)))
        adj = [[] for _ in range(n)]
        for i in range(1, n):
            adj[i].append(int(parent[i])); adj[int(parent[i])].append(i)
        diam = 0
        for s in range(n):
            dist = {s: 0}; q = [s]
            for v in q:
                for w in adj[v]:
                    if w not in dist:
                        dist[w] = dist[v] + 1; q.append(w)
            diam = max(diam, max(dist.values()))
        r = oracle.reroot(parent, [0, n])
        assert r["depth_after"][0] == (diam + 1) // 2
        _check_invariants(parent, np.array([0, n]), r)


def test_rerooted_system_has_the_permuted_solution():
    """The re-rooted arrays describe the same matrix (a symmetric permutation): Listing 2 on them gives x[perm].
    Pins perm, new_parent and usrc together: a wrong edge map changes the matrix."""
    rng = np.random.default_rng(11)
    sizes = [1, 2, 17, 64, 33]
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    parent = np.concatenate([random_parent(n, 7 + k, 0.7) for k, n in enumerate(sizes)]).astype(np.int32)
    n = int(offs[-1])
    u = -rng.uniform(0.1, 1.0, n)
    d = np.zeros(n)
    for c in range(len(sizes)):
        lo, hi = offs[c], offs[c + 1]
        for i in range(lo, hi):
            d[i] += 1.0 + abs(u[i]) * (i > lo)
            if i > lo:
                d[lo + parent[i]] += abs(u[i])
    b = rng.normal(size=n)
    x = oracle.hines_solve(parent, offs, d, u, b)
    r = oracle.reroot(parent, offs)
    x2 = oracle.hines_solve(r["new_parent"], offs, d[r["perm"]], u[r["usrc"]], b[r["perm"]])
    assert np.abs(x2 - x[r["perm"]]).max() <= 1e-12 * np.abs(x).max()
    _check_invariants(parent, offs, r)


# ---- the library's hines_reroot (csrc/reroot.cpp: centre of the tree by two breadth-first searches) against the oracle
#      (every compartment tried as the root), bit for bit --------------------------------------------------------------
def _lib_vs_oracle(parent, offs):
    import paper_1810_12742_b200 as hb
    r, o = hb.reroot(parent, offs), oracle.reroot(parent, offs)
    for a, b in (("root", "root"), ("depth_before", "depth_before"), ("depth_after", "depth_after"), ("perm", "perm"),
                 ("new_parent", "new_parent"), ("u_src", "usrc")):
        assert np.array_equal(r[a], o[b]), a
    return r


def test_library_matches_oracle_on_random_trees():
    from helpers import rooted_at
    rng = np.random.default_rng(3)
    sizes = [1, 2, 3, 5, 8, 31, 32, 33, 100, 257]
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    for trial in range(6):
        parent = np.concatenate([random_parent(n, 50 * trial + k, float(rng.uniform(0.1, 0.97))) for k, n in enumerate(sizes)]).astype(np.int32)
        _lib_vs_oracle(parent, offs)
        leafy, _, _ = rooted_at(parent, offs, lambda c, n: n - 1)       # the last compartment is always a leaf
        r = _lib_vs_oracle(leafy, offs)
        assert (r["depth_after"] <= r["depth_before"]).all()
        _check_invariants(leafy, offs, dict(r, usrc=r["u_src"]))


@pytest.mark.parametrize("cfg,scale", [(0, 1.0), (2, 0.0008), (3, 0.0004), (1, 0.0003)])
def test_library_matches_oracle_on_configs(cfg, scale):
    """The synthetic configs as generated (grown from the root: the centre is at or near the root already) and re-rooted
    at a leaf (the badly balanced case the paper has in mind)."""
    import morphgen as mg
    from helpers import rooted_at
    m = mg.make_config(cfg, scale)
    _lib_vs_oracle(m.parent, m.cell_offsets)
    leafy, _, _ = rooted_at(m.parent, m.cell_offsets, lambda c, n: n - 1)
    r = _lib_vs_oracle(leafy, m.cell_offsets)
    # a leaf's largest distance lies between the radius and the diameter of its tree
    assert ((r["depth_after"] <= r["depth_before"]) & (r["depth_before"] <= 2 * r["depth_after"])).all()
    # the plan built on the re-rooted branching cells has no more levels than the one built on the cells as given
    import paper_1810_12742_b200 as hb
    before, after = hb.Plan(leafy, m.cell_offsets), hb.Plan(r["new_parent"], m.cell_offsets)
    try:
        if cfg == 1:       # an unbranched cable rooted at its end: the middle as root halves the depth (in compartments)
            assert (r["depth_after"] == (r["depth_before"] + 1) // 2).all()      # ... and makes two branches of one
            assert after.info.max_levels == 2 and before.info.max_levels == 1
        else:
            assert after.info.max_levels <= before.info.max_levels
            if cfg == 2:
                assert after.info.max_levels < before.info.max_levels
    finally:
        before.close(); after.close()


def test_reroot_rejects_bad_input():
    import paper_1810_12742_b200 as hb
    with pytest.raises(hb.HinesError):
        hb.reroot([-1, 0, 5], [0, 3])
    with pytest.raises(hb.HinesError):
        hb.reroot([0, 0, 1], [0, 3])
    with pytest.raises(hb.HinesError):
        hb.reroot([-1, 0, 1], [0, 3, 3])
