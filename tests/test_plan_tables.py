"""CPU tests of the boundary: the library loads and exports every symbol include/hines.h declares,
hines_plan_create validates its input, its canonical tables equal the table oracle bit for bit,
and its policy tables (work items, lanes) satisfy the validity invariants of DESIGN.md
"Scheduler policy".  No compute call is made here (no GPU)."""
import ctypes
import os
import re

import numpy as np
import pytest

import morphgen as mg
import oracle
import paper_1810_12742_b200 as hb
from helpers import random_parent

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
ATOMIC = -(1 << 31)      # bit 31 of the packed descriptor word (int32)


def test_library_exports_every_declared_symbol():
    lib = hb.load_library()
    header = open(os.path.join(ROOT, "include", "hines.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(hines_[a-z_]+)\s*\(", header)))
    assert declared == sorted(hb.ABI_SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert "sm_100a" in hb.version()
    # struct sizes agree with the header's layout
    assert ctypes.sizeof(hb.Options) == 28 and ctypes.sizeof(hb.PlanInfo) == 128


def _plan_cfg(cfg, scale, **kw):
    m = mg.make_config(cfg, scale)
    return m, hb.Plan(m.parent, m.cell_offsets, **kw)


CANONICAL = ["cell_branch_offsets", "branch_start", "branch_len", "branch_parent_comp",
             "branch_parent_branch", "branch_level", "cell_nlevels", "cell_level_offsets",
             "level_count", "level_list", "child_offsets", "child_ids"]


@pytest.mark.parametrize("cfg,scale", [(0, 1.0), (1, 0.01), (2, 0.02), (3, 0.004), (4, 1.0)])
def test_canonical_tables_bit_exact(cfg, scale):
    m, plan = _plan_cfg(cfg, scale)
    T = oracle.tables(m.parent, m.cell_offsets)
    for name in CANONICAL:
        got, want = plan.table(name), getattr(T, name)
        assert got.dtype == want.dtype and np.array_equal(got, want), name
    info = plan.info
    assert info.n == m.n and info.ncells == m.ncells and info.nbranches == len(T.branch_start)
    assert info.max_levels == T.cell_nlevels.max()
    assert info.bytes_min == m.n * 32 + 4 * info.nbranches and info.bytes_literal == m.n * 36
    assert info.breadth_first == 1


def test_canonical_tables_random_topologies():
    ps = [random_parent(n, 7 * n, chain_bias=cb) for n, cb in ((1, .5), (2, .5), (3, .1), (64, .8), (257, .4), (1000, .95))]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    par = np.concatenate(ps)
    plan = hb.Plan(par, offs)
    T = oracle.tables(par, offs)
    for name in CANONICAL:
        assert np.array_equal(plan.table(name), getattr(T, name)), name
    assert plan.info.breadth_first == 0          # arbitrary p[i] < i is accepted, and reported


def test_validation_errors():
    ok_p = np.array([-1, 0, 1], np.int32)
    with pytest.raises(hb.HinesError) as e:
        hb.Plan(np.array([-1, 0, 2], np.int32), np.array([0, 3]))
    assert e.value.status == 2 and "parent[2] = 2" in str(e.value)
    with pytest.raises(hb.HinesError) as e:
        hb.Plan(np.array([0, 0, 1], np.int32), np.array([0, 3]))
    assert e.value.status == 2
    with pytest.raises(hb.HinesError) as e:          # empty cell
        hb.Plan(ok_p, np.array([0, 3, 3]))
    assert e.value.status == 2
    with pytest.raises(hb.HinesError) as e:          # offsets must start at 0
        hb.Plan(ok_p, np.array([1, 3]))
    assert e.value.status == 2
    with pytest.raises(hb.HinesError) as e:
        hb.Plan(ok_p, np.array([0, 3]), dtype=7)
    assert e.value.status == 1
    with pytest.raises(hb.HinesError) as e:
        hb.Plan(ok_p, np.array([0, 3]), threads_per_block=100)
    assert e.value.status == 1
    lib = hb.load_library()
    assert lib.hines_plan_create(None, None, 1, 0, None, None) == 1
    assert lib.hines_plan_destroy(None) == 0
    assert lib.hines_status_string(4) == b"CUDA error"


def _check_policy(m, plan, max_segment=64):
    """Validity invariants (policy-free): every branch exactly once, all branches of a resident cell
    in one item, sibling groups inside one 32-lane tile (or flagged), parents strictly on the previous
    level, segments tile every branch exactly (one separator per segment, interiors disjoint), every
    non-empty interior listed exactly once, smem need within the class, launch order a permutation."""
    T = oracle.tables(m.parent, m.cell_offsets)
    w = 8 if plan.dtype == hb.F64 else 4
    cell_item = plan.table("cell_item")
    rng_ = plan.table("item_cell_range").reshape(-1, 2)
    desc_off = plan.table("item_desc_offsets")
    lvl_off = plan.table("item_level_offsets")
    lvl_begin = plan.table("item_level_begin")
    desc = plan.table("item_desc").reshape(-1, 4)
    seg_off = plan.table("item_seg_offsets")
    segs = plan.table("item_seg").reshape(-1, 4)
    nsep_tab = plan.table("item_nsep")
    cls = plan.table("item_class")
    cls_smem = plan.table("class_smem_bytes")
    order = plan.table("item_launch_order")
    nitems = len(cls)
    assert sorted(order.tolist()) == list(range(nitems))
    assert (np.diff(cls[order]) >= 0).all()
    info = plan.info
    assert info.n_resident_items == nitems
    seen_cells = np.zeros(m.ncells, bool)
    useful = 0
    nsep_total = 0
    for it in range(nitems):
        c0, c1 = rng_[it]
        assert c1 > c0 and (cell_item[c0:c1] == it).all()
        seen_cells[c0:c1] = True
        comp0 = m.cell_offsets[c0]; n_it = m.cell_offsets[c1] - comp0
        dsc = desc[desc_off[it]:desc_off[it + 1]]
        sg = segs[seg_off[it]:seg_off[it + 1]]
        lb = lvl_begin[lvl_off[it]:lvl_off[it + 1]]
        nlev = len(lb) - 1
        assert nlev == T.cell_nlevels[c0:c1].max() and lb[0] == 0 and lb[-1] == len(dsc)
        # expected set of (end, len, pc, level)
        want = {}
        for c in range(c0, c1):
            sh = m.cell_offsets[c] - comp0
            for j in range(T.cell_branch_offsets[c], T.cell_branch_offsets[c + 1]):
                pc = T.branch_parent_comp[j]
                want[int(T.branch_start[j] + sh + T.branch_len[j] - 1)] = (
                    int(T.branch_len[j]), -1 if pc < 0 else int(pc + sh), int(T.branch_level[j]))
        got = {}
        sep_of = {}                       # separator id -> (node, top separator node or -1)
        covered = np.zeros(n_it, int)
        for l in range(nlev):
            seg_l = dsc[lb[l]:lb[l + 1]]
            nseg = seg_l[:, 1] & 0xfffff
            sj = (seg_l[:, 1] >> 20) & 0x7ff
            real = nseg > 0
            for (end, word, pc, sbase), ns, s_ in zip(seg_l[real], nseg[real], sj[real]):
                ln, pcw, lw = want[int(end)]
                assert int(end) not in got and pcw == pc and lw == l
                got[int(end)] = 1
                assert ns == -(-ln // max_segment) and s_ == -(-ln // ns)
                start = end - ln + 1
                for k in range(ns):
                    b = end - k * s_
                    a = max(start, b - s_ + 1)
                    t = b - s_ if k < ns - 1 else pc
                    assert (sbase + k) not in sep_of
                    sep_of[int(sbase + k)] = (int(a), int(b - a), int(t))
                    covered[a:b + 1] += 1
            pcs = seg_l[:, 2]
            for pcv in np.unique(pcs[real & (pcs >= 0)]):
                idx = np.nonzero(real & (pcs == pcv))[0]
                flagged = seg_l[idx, 1] < 0
                if flagged.any():
                    assert flagged.all() and len(idx) > 32
                else:
                    assert idx.min() // 32 == idx.max() // 32 and (np.diff(idx) == 1).all()
        assert set(got) == set(want) and (covered == 1).all()
        assert nsep_tab[it] == len(sep_of) and sorted(sep_of) == list(range(len(sep_of)))
        # parents are separators of the level above
        ends_level = {e: v[2] for e, v in want.items()}
        for e, (ln, pc, l) in want.items():
            if pc >= 0:
                assert ends_level[pc] == l - 1
        # segment lane list: exactly the non-empty interiors, once each
        real = sg[:, 1] > 0
        listed = {int(sid): (int(a), int(mm), int(t)) for a, mm, t, sid in sg[real]}
        assert len(listed) == real.sum()
        assert listed == {k: v for k, v in sep_of.items() if v[1] > 0}
        useful += int(sg[real, 1].sum())
        nsep_total += len(sep_of)
        # wavefront groups (16 lanes fp64 / 32 lanes fp32) mostly have distinct start residues
        R = 128 // w
        # shared-memory need within the class
        E = 16 // w
        L = -(-(comp0 % E + n_it) // E) * E
        meta = -(-(nlev + 1) // 4) * 4 + 4 * len(dsc) + 4 * len(sg)
        assert 16 + 3 * L * w + 2 * (-(-len(sep_of) // E) * E) * w + 4 * meta <= cls_smem[cls[it]] <= 232448
    assert (seen_cells == (cell_item >= 0)).all()
    # streaming path: every branch of every non-resident cell exactly once, children complete
    sd = plan.table("stream_desc").reshape(-1, 6)
    sl = plan.table("stream_level_begin")
    sc = plan.table("stream_child").reshape(-1, 2)
    stream_cells = np.nonzero(cell_item < 0)[0]
    assert info.n_stream_cells == len(stream_cells)
    want = {}
    for c in stream_cells:
        o = m.cell_offsets[c]
        for j in range(T.cell_branch_offsets[c], T.cell_branch_offsets[c + 1]):
            pc = T.branch_parent_comp[j]
            want[int(o + T.branch_start[j])] = (int(T.branch_len[j]), -1 if pc < 0 else int(o + pc), int(T.branch_level[j]),
                                                int(T.child_offsets[j + 1] - T.child_offsets[j]))
    assert len(sd) == len(want) == info.n_stream_branches
    ws_seen = set()
    for l in range(len(sl) - 1):
        seg = sd[sl[l]:sl[l + 1]]
        assert (np.diff(seg[:, 1]) <= 0).all()                         # length descending (S7)
        for gs, ln, gp, ws, cb, nchild in seg:
            assert want[int(gs)] == (int(ln), int(gp), l, int(nchild))
            assert ws not in ws_seen; ws_seen.add(int(ws))
            for k in range(nchild):
                cgs, cws = sc[cb + k]
                assert want[int(cgs)][1] == gs + ln - 1 and want[int(cgs)][2] == l + 1
                assert cws - ws == cgs - gs                           # same cell, same shift
            useful += int(ln)
    assert useful + nsep_total == m.n and useful == info.useful_lane_steps
    assert info.n_resident_unknowns + info.n_stream_unknowns == m.n
    assert info.padded_lane_steps >= useful


@pytest.mark.parametrize("cfg,scale,kw", [
    (0, 1.0, {}), (0, 1.0, dict(policy_flags=hb.POLICY_NO_GROUPING)),
    (2, 0.004, {}), (2, 0.004, dict(smem_bytes_per_block=60000)),
    (2, 0.003, dict(policy_flags=hb.POLICY_FORCE_STREAM)),
    (3, 0.002, {}), (3, 0.002, dict(dtype=hb.F32)), (1, 0.002, {}), (1, 0.002, dict(max_segment=7)),
    (2, 0.003, dict(max_segment=2)), (3, 0.002, dict(max_segment=16)),
])
def test_policy_tables_valid(cfg, scale, kw):
    m, plan = _plan_cfg(cfg, scale, **kw)
    _check_policy(m, plan, kw.get("max_segment", 64))


def test_policy_star_with_many_siblings_and_odd_offsets():
    star = np.array([-1] + [0] * 70, np.int32)                        # 70 siblings: group spans tiles -> flagged
    ps = [star, random_parent(33, 1), np.array([-1], np.int32), random_parent(200, 2, .7), star[:40]]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    m = mg.Morphology(np.concatenate(ps), offs)
    for kw in ({}, dict(dtype=hb.F32), dict(policy_flags=hb.POLICY_NO_GROUPING)):
        plan = hb.Plan(m.parent, m.cell_offsets, **kw)
        _check_policy(m, plan)
        assert (plan.table("item_desc").reshape(-1, 4)[:, 1] < 0).any()


def test_config4_goes_to_streaming_path_and_grouping_is_greedy_in_order():
    m, plan = _plan_cfg(4, 1.0)
    info = plan.info
    assert info.n_stream_cells == 1 and info.n_resident_items == 0 and plan.launches_per_solve == 34
    # config 0: 64 cells x 75 unknowns: greedy contiguous groups up to 56 KiB
    m, plan = _plan_cfg(0, 1.0)
    r = plan.table("item_cell_range").reshape(-1, 2)
    assert r[0, 0] == 0 and r[-1, 1] == 64 and (r[1:, 0] == r[:-1, 1]).all()
    assert plan.info.n_stream_cells == 0 and len(r) < 64


def test_solve_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    m, plan = _plan_cfg(0, 1.0)
    x = np.zeros(m.n)
    with pytest.raises(hb.HinesError) as e:
        plan.solve_host(x, x, x, x.copy())
    assert e.value.status == 4 and "no CPU fallback" in str(e.value)
