"""f1: the paper's branch splitting pass.  The split oracle (oracle/split_oracle.c) is pinned by a
hand-worked example, closed forms and invariants; the plan's HINES_TABLE_SPLIT_* tables must equal it bit for bit;
with HINES_POLICY_SPLIT_LEVEL_MEAN the plan's segments follow those pieces."""
import json
import os

import numpy as np
import pytest

import morphgen as mg
import oracle
import paper_1810_12742_b200 as hb
from helpers import random_parent
from plan_interpreter import parts_of

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "split_example.json")))
NAMES = ("piece_offsets", "piece_len", "piece_level", "level_stat")


@pytest.mark.parametrize("case", ["one_cell", "two_cells"])
def test_hand_worked_example(case):
    g = GOLD[case]
    par = np.array(GOLD["parent_cell"] + ([-1] if case == "two_cells" else []), np.int32)
    got = oracle.level_mean_split(par, np.array(g["cell_offsets"], np.int64))
    for name, a in zip(NAMES, got):
        assert a.tolist() == g[name], name
    plan = hb.Plan(par, np.array(g["cell_offsets"], np.int64))
    for name in NAMES:
        assert plan.table("split_" + name).tolist() == g[name], name


def test_closed_forms():
    # equal lengths on every level: nothing is longer than the average, nothing is cut (configs 0, 1, 4)
    for cfg, scale in ((0, 1.0), (1, 0.005), (4, 1.0)):
        m = mg.make_config(cfg, scale)
        offs, ln, lv, stat = oracle.level_mean_split(m.parent, m.cell_offsets)
        T = oracle.tables(m.parent, m.cell_offsets)
        assert np.array_equal(np.diff(offs), np.ones(len(T.branch_len))) and np.array_equal(ln, T.branch_len)
        assert np.array_equal(lv, T.branch_level)
    # one cable of n among k-1 cables of one compartment: c = ceil((n + k - 1) / k) on level 0, then the rest alone
    n, k = 100, 5
    par = np.concatenate([np.arange(-1, n - 1), -np.ones(k - 1)]).astype(np.int32)
    offs = np.concatenate([[0, n], n + 1 + np.arange(k - 1)]).astype(np.int64)
    po, ln, lv, stat = oracle.level_mean_split(par, offs)
    c = -(-(n + k - 1) // k)
    assert ln[:2].tolist() == [c, n - c] and lv[:2].tolist() == [0, 1] and stat.tolist() == [n + k - 1, k, n - c, 1]


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_invariants_random_trees(seed):
    ps = [random_parent(n, seed * 100 + n, cb) for n, cb in ((40, .5), (300, .8), (7, .2), (1000, .95), (1, .5))]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])]).astype(np.int64)
    par = np.concatenate(ps)
    po, ln, lv, stat = oracle.level_mean_split(par, offs)
    T = oracle.tables(par, offs)
    nb = len(T.branch_len)
    assert len(po) == nb + 1 and (ln >= 1).all()
    cut = -(-stat[0::2] // stat[1::2])
    for j in range(nb):
        pl, pv = ln[po[j]:po[j + 1]], lv[po[j]:po[j + 1]]
        assert pl.sum() == T.branch_len[j], "pieces tile the branch"
        assert (np.diff(pv) == 1).all(), "a rest sits one level below its head"
        assert (pl <= cut[pv]).all() and (pl[:-1] == cut[pv[:-1]]).all(), "a head has exactly ceil(mean) compartments"
    # a child's first piece sits one level below its parent's last: levels shift by the cuts above
    for c in range(len(ps)):
        b0 = T.cell_branch_offsets[c]
        for j in range(b0, T.cell_branch_offsets[c + 1]):
            pb = T.branch_parent_branch[j]
            first = lv[po[j]]
            if pb < 0:
                assert first == 0
            else:
                assert first == lv[po[b0 + pb + 1] - 1] + 1
                cuts_above, a = 0, j
                while T.branch_parent_branch[a] >= 0:
                    a = b0 + T.branch_parent_branch[a]
                    cuts_above += po[a + 1] - po[a] - 1
                assert first == T.branch_level[j] + cuts_above
    # the statistics are those of the pieces before cutting: recompute them from the result
    for L in range(len(cut)):
        on = np.nonzero(lv == L)[0]
        rest = np.array([ln[k:po[np.searchsorted(po, k, side="right")]].sum() for k in on])
        assert rest.sum() == stat[2 * L] and len(on) == stat[2 * L + 1]


@pytest.mark.parametrize("cfg,scale", [(0, 1.0), (1, 0.01), (2, 0.02), (3, 0.004), (4, 1.0)])
def test_plan_split_tables_bit_exact(cfg, scale):
    m = mg.make_config(cfg, scale)
    want = oracle.level_mean_split(m.parent, m.cell_offsets)
    plan = hb.Plan(m.parent, m.cell_offsets)
    for name, a in zip(NAMES, want):
        got = plan.table("split_" + name)
        assert got.dtype == a.dtype and np.array_equal(got, a), name


def test_policy_level_mean_segments_follow_the_pieces():
    """With the flag and max_segment = 1023 the plan's segments are exactly the paper's pieces, and the tables still
    solve the systems (tests/plan_interpreter.py)."""
    from test_plan_tables import _check_interpreted
    m = mg.make_config(2, 0.004)
    po, ln, lv, stat = oracle.level_mean_split(m.parent, m.cell_offsets)
    plan = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_SPLIT_LEVEL_MEAN, max_segment=1023)
    nseg = sum(int((~p.ghost[:p.h["nlevnode"]]).sum()) for p in parts_of(plan))
    assert nseg == len(ln) and plan.info.n_stream_cells == 0
    assert plan.info.useful_lane_steps == m.n - len(ln)
    _check_interpreted(m, plan)
    plan = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_SPLIT_LEVEL_MEAN)     # pieces bounded by max_segment too
    _check_interpreted(m, plan)


# ---- f4 ("more local heuristics, like per block averages"): the same rule with the level means taken over
#      the cells of one block.  Oracle = oracle_level_mean_split applied to the cells of every work item on their own -----
def _block_mean_pieces(m, plan):
    """Per global branch the pieces the ORACLE gives when each item's cells are split as a batch of their own."""
    t = oracle.tables(m.parent, m.cell_offsets)
    item_cells, item_offs = plan.table("item_cells"), plan.table("item_cell_offsets")
    want_len = [None] * len(t.branch_len)
    want_lev = [None] * len(t.branch_len)
    seen = np.zeros(m.ncells, bool)
    for it in range(len(item_offs) - 1):
        cells = item_cells[item_offs[it]:item_offs[it + 1]]
        seen[cells] = True
        par = np.concatenate([m.parent[m.cell_offsets[c]:m.cell_offsets[c + 1]] for c in cells])
        offs = np.concatenate([[0], np.cumsum([m.cell_offsets[c + 1] - m.cell_offsets[c] for c in cells])]).astype(np.int64)
        po, ln, lv, _ = oracle.level_mean_split(par, offs)
        gbr = np.concatenate([np.arange(t.cell_branch_offsets[c], t.cell_branch_offsets[c + 1]) for c in cells])
        for k, j in enumerate(gbr):
            want_len[j], want_lev[j] = ln[po[k]:po[k + 1]], lv[po[k]:po[k + 1]]
    for c in np.nonzero(~seen)[0]:                        # cells of the streaming path: uncut
        for j in range(t.cell_branch_offsets[c], t.cell_branch_offsets[c + 1]):
            want_len[j], want_lev[j] = np.array([t.branch_len[j]], np.int32), np.array([t.branch_level[j]], np.int32)
    return want_len, want_lev


@pytest.mark.parametrize("cfg,scale,kw", [(0, 1.0, {}), (3, 0.004, {}), (2, 0.004, {}), (3, 0.004, dict(group_smem_bytes=20000)),
                                          (2, 0.002, dict(smem_bytes_per_block=48000, cluster_max=2, split_smem_bytes=20000)),
                                          (1, 0.004, {})])
def test_policy_block_mean_tables_bit_exact_and_solve(cfg, scale, kw):
    from test_plan_tables import _check_interpreted
    m = mg.make_config(cfg, scale)
    plan = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_SPLIT_BLOCK_MEAN, **kw)
    want_len, want_lev = _block_mean_pieces(m, plan)
    po, ln, lv = plan.table("split_piece_offsets"), plan.table("split_piece_len"), plan.table("split_piece_level")
    assert len(po) == len(want_len) + 1 and len(plan.table("split_level_stat")) == 0
    for j in range(len(want_len)):
        assert np.array_equal(ln[po[j]:po[j + 1]], want_len[j]) and np.array_equal(lv[po[j]:po[j + 1]], want_lev[j]), j
    _check_interpreted(m, plan)                            # the segments follow these pieces and the tables solve the systems
    # a block's own means differ from the batch's (unless all cells are alike): the heterogeneous config must show it
    if cfg == 3 and not kw:
        glob = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_SPLIT_LEVEL_MEAN)
        assert not np.array_equal(glob.table("split_piece_len"), ln)


def test_block_mean_of_one_block_is_the_level_mean():
    """Closed form: when the whole batch is one block, block means = batch means."""
    m = mg.make_config(0, 0.25)                            # 16 cells of 75 unknowns: one group
    a = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_SPLIT_BLOCK_MEAN)
    b = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_SPLIT_LEVEL_MEAN)
    assert a.info.n_resident_items == 1 and b.info.n_resident_items == 1
    for name in ("split_piece_offsets", "split_piece_len", "split_piece_level"):
        assert np.array_equal(a.table(name), b.table(name))
    assert np.array_equal(a.table("part_meta"), b.table("part_meta"))
