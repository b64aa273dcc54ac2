"""Pins for oracle/tables_oracle.c: closed forms for the regular configs (tests/golden/
fig21_tables.json), the merge example of reading S4, and a pure-Python brute
force that derives branches, levels and lists a different way (chains of only-children,
levels by walking to the root)."""
import json
import os

import numpy as np
import pytest

import morphgen as mg
import oracle
from helpers import random_parent

GOLDEN = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "fig21_tables.json")))


def brute_tables(p):
    """Slow, different-in-structure derivation for ONE cell."""
    n = len(p)
    kids = [[] for _ in range(n)]
    for i in range(1, n):
        kids[p[i]].append(i)
    # i continues its parent's branch iff it is the only child and numbered right after it
    cont = [False] * n
    for i in range(1, n):
        cont[i] = (len(kids[p[i]]) == 1 and p[i] == i - 1)
    starts = [i for i in range(n) if not cont[i]]
    sid = {s: j for j, s in enumerate(starts)}
    head = [0] * n                      # first compartment of the branch of i
    for i in range(n):
        head[i] = head[i - 1] if cont[i] else i
    length = [sum(1 for i in range(n) if head[i] == s) for s in starts]
    pcomp = [-1 if s == 0 else int(p[s]) for s in starts]
    pbr = [-1 if s == 0 else sid[head[p[s]]] for s in starts]
    level = []
    for s in starts:                    # count branch changes on the way to the root
        l, v = 0, s
        while v != 0:
            v = head[p[v]]
            l += 1
        level.append(l)
    nlev = max(level) + 1
    count = [level.count(l) for l in range(nlev)]
    lst = sorted(range(len(starts)), key=lambda j: (level[j], -length[j], j))
    children = [[c for c in range(len(starts)) if pbr[c] == j] for j in range(len(starts))]
    return dict(start=starts, length=length, pcomp=pcomp, pbr=pbr, level=level, count=count,
                lst=lst, children=children)


def check_cell(T, c, ref):
    b0, b1 = T.cell_branch_offsets[c], T.cell_branch_offsets[c + 1]
    assert list(T.branch_start[b0:b1]) == ref["start"]
    assert list(T.branch_len[b0:b1]) == ref["length"]
    assert list(T.branch_parent_comp[b0:b1]) == ref["pcomp"]
    assert list(T.branch_parent_branch[b0:b1]) == ref["pbr"]
    assert list(T.branch_level[b0:b1]) == ref["level"]
    l0, l1 = T.cell_level_offsets[c], T.cell_level_offsets[c + 1]
    assert T.cell_nlevels[c] == len(ref["count"]) == l1 - l0
    assert list(T.level_count[l0:l1]) == ref["count"]
    assert list(T.level_list[b0:b1]) == ref["lst"]
    for j in range(b1 - b0):
        ch = T.child_ids[T.child_offsets[b0 + j]:T.child_offsets[b0 + j + 1]]
        assert list(ch) == ref["children"][j]


def test_config0_closed_form():
    g = GOLDEN["config0"]
    m = mg.make_config(0)
    assert list(m.parent[:12]) == g["parent_first12"]
    T = oracle.tables(m.parent, m.cell_offsets)
    assert len(T.branch_start) == 64 * g["nbranches"]
    for c in (0, 17, 63):
        b0 = T.cell_branch_offsets[c]; s = slice(b0, b0 + 15)
        assert list(T.branch_start[s]) == g["branch_start"]
        assert (T.branch_len[s] == g["branch_len"]).all()
        assert list(T.branch_parent_comp[s]) == g["branch_parent_comp"]
        assert list(T.branch_parent_branch[s]) == g["branch_parent_branch"]
        assert list(T.branch_level[s]) == g["branch_level"]
        assert list(T.level_count[T.cell_level_offsets[c]:T.cell_level_offsets[c + 1]]) == g["level_count"]
        assert list(T.level_list[s]) == list(range(15))      # equal lengths: ties by id


def test_merge_example():
    g = GOLDEN["merge_example"]
    p = np.array(g["p"], np.int32)
    T = oracle.tables(p, np.array([0, len(p)]))
    assert list(T.branch_start) == g["branch_start"]
    assert list(T.branch_len) == g["branch_len"]
    assert list(T.branch_parent_comp) == g["branch_parent_comp"]
    assert list(T.branch_level) == g["branch_level"]
    # a single child numbered right after its parent merges: plain cable = one branch
    T = oracle.tables(np.arange(-1, 9, dtype=np.int32), np.array([0, 10]))
    assert list(T.branch_start) == [0] and list(T.branch_len) == [10]
    # a single child NOT numbered right after its parent is its own branch
    T = oracle.tables(np.array([-1, 0, 0, 2, 1], np.int32), np.array([0, 5]))
    assert list(T.branch_start) == [0, 1, 2, 4] and list(T.branch_len) == [1, 1, 2, 1]
    assert list(T.branch_level) == [0, 1, 1, 2]


def test_config1_and_4_closed_forms():
    m = mg.make_config(1, 0.001)
    T = oracle.tables(m.parent, m.cell_offsets)
    assert (T.branch_len == 1000).all() and (T.cell_nlevels == 1).all() and len(T.child_ids) == 0
    m = mg.make_config(4)
    T = oracle.tables(m.parent, m.cell_offsets)
    nb = 131071
    assert len(T.branch_start) == nb and m.n == 1310710
    j = np.arange(nb)
    assert (T.branch_start == 10 * j).all() and (T.branch_len == 10).all()
    assert (T.branch_parent_branch[1:] == (j[1:] - 1) // 2).all()
    assert (T.branch_parent_comp[1:] == 10 * ((j[1:] - 1) // 2) + 9).all()
    assert (T.branch_level == np.floor(np.log2(j + 1)).astype(int)).all()
    assert list(T.level_count) == [1 << l for l in range(17)]
    assert (T.child_ids == j[1:]).all() and (np.diff(T.child_offsets)[:65535] == 2).all()


@pytest.mark.parametrize("seed", range(6))
def test_brute_force_random(seed):
    ps = [random_parent(n, 100 * seed + n, chain_bias=cb) for n, cb in ((1, .5), (2, .5), (40, .8), (63, .3), (150, .9))]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    T = oracle.tables(np.concatenate(ps), offs)
    for c, p in enumerate(ps):
        check_cell(T, c, brute_tables(p))


def test_brute_force_generator_cells():
    m = mg.make_config(2, 0.0005)      # 5 random dendrites
    T = oracle.tables(m.parent, m.cell_offsets)
    for c in range(m.ncells):
        check_cell(T, c, brute_tables(m.parent[m.cell_offsets[c]:m.cell_offsets[c + 1]]))
    # generator intent vs canonical rule: only merges (S4) may reduce the count
    assert len(T.branch_start) <= len(m.gen_branch_len)
    assert T.branch_len.sum() == m.n


def test_structural_invariants():
    """Every non-root branch hangs off the LAST compartment of its parent branch and
    parent_branch < branch id (consequence of S4 + p[i] < i)."""
    m = mg.make_config(3, 0.002)
    T = oracle.tables(m.parent, m.cell_offsets)
    cell = np.repeat(np.arange(m.ncells), np.diff(T.cell_branch_offsets))
    nonroot = T.branch_parent_branch >= 0
    pb_glob = T.cell_branch_offsets[cell] + T.branch_parent_branch
    assert (T.branch_parent_branch[nonroot] < (np.arange(len(cell)) - T.cell_branch_offsets[cell])[nonroot]).all()
    last = T.branch_start[pb_glob[nonroot]] + T.branch_len[pb_glob[nonroot]] - 1
    assert (T.branch_parent_comp[nonroot] == last).all()


def test_malformed_rejected():
    with pytest.raises(ValueError):
        oracle.tables(np.array([-1, 1], np.int32), np.array([0, 2]))
    with pytest.raises(ValueError):
        oracle.tables(np.array([0, 0], np.int32), np.array([0, 2]))
