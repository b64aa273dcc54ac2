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
from plan_interpreter import parts_of, segments

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


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
    assert ctypes.sizeof(hb.Options) == 40 and ctypes.sizeof(hb.PlanInfo) == 184


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




def _pieces_fixed(ln, S):
    """Pieces of a branch of ln compartments under the fixed-bound rule, top-down (P4)."""
    nseg = max(1, (5 * ln + 2 * S) // (5 * S))             # len / max_segment + 0.4, cut off
    sj = -(-ln // nseg)
    if nseg > 1 and sj % 2 == 0:
        sj += 1                                            # odd: the segments of a branch start on distinct banks
    nseg = -(-ln // sj)                                    # no empty segment
    return [ln - (nseg - 1) * sj] + [sj] * (nseg - 1)


def _check_policy(m, plan, max_segment=0):
    """Validity invariants (policy-free): every cell in exactly one on-chip item or on the streaming path; the runs of
    an item's parts tile the compartments of its cells exactly once; segments tile every branch exactly, in the
    pieces the written rule gives, each listed once; a segment's upper node is the node of the compartment above it
    (a ghost parent when that compartment lives in another part); every node once on the level of its depth,
    children consecutive behind their parent; exports and ghost children pair up one to one; shared-memory need
    within the class; every part launched exactly once per phase."""
    T = oracle.tables(m.parent, m.cell_offsets)
    w = 8 if plan.dtype == hb.F64 else 4
    E = 16 // w
    cell_item = plan.table("cell_item")
    co, cells = plan.table("item_cell_offsets"), plan.table("item_cells")
    kind = plan.table("item_kind")
    poff = plan.table("item_part_offsets")
    cls = plan.table("item_class")
    cls_smem, cls_cluster = plan.table("class_smem_bytes"), plan.table("class_cluster")
    cls_threads, cls_phase = plan.table("class_threads"), plan.table("class_phase")
    cfirst, ccount, cparts = plan.table("class_first"), plan.table("class_count"), plan.table("class_parts")
    order = plan.table("item_launch_order")
    parts = parts_of(plan)
    nitems = len(kind)
    info = plan.info
    assert sorted(order.tolist()) == list(range(nitems))
    assert ((cls_threads % 32 == 0) & (cls_threads >= 32) & (cls_threads <= 1024)).all()
    assert info.n_resident_items == nitems and info.n_parts == len(parts) and info.n_blocks == len(cparts)
    # launches: every part of an ordinary item once; a split item's sub-tree parts in phases A and C, its top in B
    launched = {}
    for q in range(len(cfirst)):
        ids = cparts[cfirst[q]:cfirst[q] + ccount[q]]
        assert ccount[q] % cls_cluster[q] == 0
        for k, pid in enumerate(ids):
            h = parts[pid].h
            launched.setdefault(int(pid), []).append(int(cls_phase[q]))
            need = 16 + 512 + 6 * w * (-(-(h["nnode"] + 1) // E) * E) + 4 * h["meta_len"] + (4 if parts[pid].factored else 3) * w * h["L"]
            assert need <= cls_smem[q] <= 232448
            assert h["maxwidth"] <= cls_threads[q] or True
            if cls_cluster[q] > 1:
                assert h["rank"] == k % cls_cluster[q] and kind[h["item"]] == 1
    useful = 0
    nsep_total = 0
    seen_cells = np.zeros(m.ncells, bool)
    for it in range(nitems):
        cs = cells[co[it]:co[it + 1]]
        assert len(cs) > 0 and (np.diff(cs) > 0).all() and (cell_item[cs] == it).all()
        assert not seen_cells[cs].any()
        seen_cells[cs] = True
        ps = parts[poff[it]:poff[it + 1]]
        assert (kind[it] == 0) == (len(ps) == 1) and (kind[it] == 0 or len(cs) == 1)
        for r, p in enumerate(ps):
            want_ph = [0] if kind[it] != 2 else ([2] if r == 0 else [1, 3])
            assert launched[poff[it] + r] == want_ph
        S_it = max_segment if max_segment else (40 if kind[it] == 0 else 64)
        # compartments -> (part, staged index); runs tile the item's cells exactly once
        where = {}
        for r, p in enumerate(ps):
            for g, ln, so, _ in p.runs:
                for k in range(int(ln)):
                    assert int(g) + k not in where
                    where[int(g) + k] = (r, int(so) + k)
        want_comps = np.concatenate([np.arange(m.cell_offsets[c], m.cell_offsets[c + 1]) for c in cs])
        assert sorted(where) == want_comps.tolist()
        # segments of every part: separator position -> node
        node_at = {}                                       # global compartment -> (part, node)
        seg_at = {}                                        # global first compartment -> (part, interior, node, tnode)
        for r, p in enumerate(ps):
            inv = {v: k for k, (pr, v) in where.items() if pr == r}
            seen_nodes = set()
            for a, lens, node, tnode in segments(p.seg):
                mm = sum(lens) + max(0, len(lens) - 1)
                assert 0 <= node < p.h["nlevnode"] and node not in seen_nodes and not p.ghost[node]
                seen_nodes.add(node)
                g0 = inv[a]
                assert all(inv[a + k] == g0 + k for k in range(mm + 1)), "a segment is contiguous in memory and in the staging"
                seg_at[g0] = (r, mm, node, tnode)
                node_at[g0 + mm] = (r, node)
                useful += mm
            assert len(seen_nodes) == int((~p.ghost[:p.h["nlevnode"]]).sum())
            nsep_total += len(seen_nodes)
        # branches: the written pieces, one segment each, chained from the top; the node above a branch's first
        # piece is the node of its parent compartment, through a ghost parent when that lives in part 0
        level_of = []
        for p in ps:
            lv = np.zeros(p.h["nlevnode"], int)
            if not p.chains:
                for l in range(p.h["nlev"]):
                    lv[p.lb[l]:p.lb[l + 1]] = l
            level_of.append(lv)
        exports = {(r, int(e[0])): e for r, p in enumerate(ps) for e in p.exps}
        n_exp_seen = 0
        for c in cs:
            o = int(m.cell_offsets[c])
            for j in range(T.cell_branch_offsets[c], T.cell_branch_offsets[c + 1]):
                start, ln, pc = o + int(T.branch_start[j]), int(T.branch_len[j]), int(T.branch_parent_comp[j])
                prev = None if pc < 0 else node_at[o + pc]
                pos = start
                for k, plen in enumerate(_pieces_fixed(ln, S_it)):
                    r, mm, node, tnode = seg_at[pos]
                    p = ps[r]
                    assert mm == plen - 1, (it, j, k)
                    if prev is None:
                        assert tnode == -1 and p.pnode[node] == node
                    elif prev[0] == r:
                        assert tnode == prev[1] and p.pnode[node] == prev[1]
                        if not p.chains:
                            assert level_of[r][node] == level_of[r][prev[1]] + 1
                            assert node in p.children(prev[1], w)
                    else:                                      # an exported sub-tree root
                        assert k == 0 and r > 0 and prev[0] == 0
                        e = exports[(r, node)]
                        assert tnode == e[1] >= p.h["nlevnode"] and p.pnode[node] == e[1]
                        gl = [g for g in ps[0].ghosts if g[1] == e[2]] if kind[it] == 2 else [g for g in ps[0].ghosts if g[0] == e[2]]
                        assert len(gl) == 1 and gl[0][2] == prev[1] and ps[0].ghost[gl[0][0]]
                        assert int(gl[0][0]) in ps[0].children(prev[1], w)
                        # cluster items: the ghost child's entry names where rank 0 sends the parent's x (checked word by
                        # word in plan_interpreter.solve_with_tables); split items go through the exchange buffer
                        assert (int(gl[0][3]) >> 20) == (r if kind[it] == 1 else 0) and (kind[it] == 1 or gl[0][3] == 0)
                        n_exp_seen += 1
                    prev = (r, node)
                    pos += plen
                assert pos == start + ln
        assert n_exp_seen == sum(p.h["nexp"] for p in ps) == ps[0].h["nghost"]
        for p in ps:                                           # every child listed belongs to its parent
            if p.chains:
                continue
            assert p.h["maxwidth"] == max([0] + [int(p.lb[l + 1] - p.lb[l]) for l in range(p.h["nlev"])])
            nkids = 0
            for v in range(p.h["nlevnode"]):
                if not p.ghost[v]:
                    for ch in p.children(v, w):
                        assert p.ghost[ch] or p.pnode[ch] == v
                        nkids += 1
            roots = sum(1 for v in range(p.h["nlevnode"]) if not p.ghost[v] and (p.pnode[v] == v or p.pnode[v] >= p.h["nlevnode"]))
            assert nkids + roots == p.h["nlevnode"]
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


def _check_interpreted(m, plan):
    """The tables, executed lane by lane on the CPU (tests/plan_interpreter.py), solve the systems."""
    from plan_interpreter import solve_with_tables
    d, u, b = mg.system(m)
    x = solve_with_tables(plan, m, d, u, b)
    xr = oracle.hines_solve(m.parent, m.cell_offsets, d, u, b)
    sel = np.repeat(plan.table("cell_item") >= 0, np.diff(m.cell_offsets))
    assert np.isfinite(x[sel]).all() and np.isnan(x[~sel]).all()
    if sel.any():
        assert np.abs(x[sel] - xr[sel]).max() < 1e-12


@pytest.mark.parametrize("cfg,scale,kw", [
    (0, 1.0, {}), (0, 1.0, dict(policy_flags=hb.POLICY_NO_GROUPING)),
    (2, 0.004, {}), (2, 0.004, dict(smem_bytes_per_block=60000, policy_flags=hb.POLICY_NO_CLUSTER)),
    (2, 0.003, dict(policy_flags=hb.POLICY_FORCE_STREAM)),
    (3, 0.002, {}), (3, 0.002, dict(dtype=hb.F32)), (1, 0.002, {}), (1, 0.002, dict(max_segment=7)),
    (1, 0.002, dict(policy_flags=hb.POLICY_NO_PCR)), (3, 0.002, dict(policy_flags=hb.POLICY_INPUT_ORDER)),
    (2, 0.003, dict(max_segment=2)), (3, 0.002, dict(max_segment=16)),
    (2, 0.004, dict(chunk_smem_bytes=30000, cluster_max=16)), (1, 0.002, dict(max_segment=5, chunk_smem_bytes=8000)),
    (3, 0.002, dict(chunk_smem_bytes=40000, cluster_max=4)),
    (2, 0.002, dict(chunk_smem_bytes=20000, cluster_max=2, split_smem_bytes=20000)),
    (2, 0.004, dict(smem_bytes_per_block=48000, cluster_max=2, split_smem_bytes=20000)),
    (2, 0.004, dict(smem_bytes_per_block=64000, cluster_max=2, split_smem_bytes=12000, max_segment=9)),
])
def test_policy_tables_valid(cfg, scale, kw):
    m, plan = _plan_cfg(cfg, scale, **kw)
    _check_policy(m, plan, kw.get("max_segment", 0))
    _check_interpreted(m, plan)


def test_policy_star_with_many_siblings_and_odd_offsets():
    star = np.array([-1] + [0] * 70, np.int32)                        # 70 siblings: beyond the two child slots -> the loop
    ps = [star, random_parent(33, 1), np.array([-1], np.int32), random_parent(200, 2, .7), star[:40],
          random_parent(1001, 3, .97)]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    m = mg.Morphology(np.concatenate(ps), offs)
    for kw in ({}, dict(dtype=hb.F32), dict(policy_flags=hb.POLICY_NO_GROUPING), dict(max_segment=3),
               dict(chunk_smem_bytes=6000, max_segment=4)):
        plan = hb.Plan(m.parent, m.cell_offsets, **kw)
        _check_policy(m, plan, kw.get("max_segment", 0))
        _check_interpreted(m, plan)
        assert max(int(p.nc.max()) for p in parts_of(plan)) == 70    # the star's root pulls its 70 children


def test_clusters_take_the_cells_too_large_for_one_block():
    m, plan = _plan_cfg(3, 0.004)
    info = plan.info
    assert info.n_cluster_cells > 0 and info.n_stream_cells == 0 and info.n_split_cells == 0
    cl = plan.table("class_cluster")
    assert cl.min() == 1 and cl.max() <= 16 and (np.diff(cl) <= 0).all()
    m, plan = _plan_cfg(3, 0.004, policy_flags=hb.POLICY_POW2_CLUSTERS)
    assert set(plan.table("class_cluster").tolist()) <= {1, 2, 4, 8, 16}
    m, plan = _plan_cfg(3, 0.004, policy_flags=hb.POLICY_NO_CLUSTER)
    assert plan.info.n_cluster_cells == 0 and (plan.table("class_cluster") == 1).all()


def test_config4_is_a_split_item_and_grouping_is_greedy_in_order():
    """Config 4 (one cell of 1.3 M unknowns, beyond any cluster) runs as a split item: sub-tree parts backward, the
    top part, the sub-tree parts again -- three launches, no streaming path."""
    m, plan = _plan_cfg(4, 1.0)
    info = plan.info
    assert info.n_split_cells == 1 and info.n_stream_cells == 0 and info.n_resident_items == 1
    assert plan.table("class_phase").tolist() == [1, 2, 3] and plan.launches_per_solve == 3
    assert info.n_exports == info.n_parts - 1 == 512
    _check_policy(m, plan)
    m, plan = _plan_cfg(4, 1.0, policy_flags=hb.POLICY_NO_SPLIT)
    assert plan.info.n_stream_cells == 1 and plan.launches_per_solve == 34
    # config 0: 64 cells x 75 unknowns: greedy groups in input order up to 56 KiB
    m, plan = _plan_cfg(0, 1.0)
    co, cells = plan.table("item_cell_offsets"), plan.table("item_cells")
    assert cells.tolist() == list(range(64)) and plan.info.n_stream_cells == 0 and len(co) - 1 < 64


def test_long_root_branch_with_a_fork_takes_a_correct_path():
    """a very long root branch (thousands of reduced nodes) with a fork at its end.  Whatever path the
    plan picks, the tables must solve the system (no descriptor field may wrap)."""
    n = 20000
    p = np.arange(-1, n + 1, dtype=np.int32)
    p[n + 1] = n - 1                                                  # two children at the end of the root branch
    m = mg.Morphology(p, np.array([0, n + 2], np.int64))
    for kw in (dict(max_segment=8), dict(max_segment=8, dtype=hb.F32), {}):
        plan = hb.Plan(m.parent, m.cell_offsets, **kw)
        _check_interpreted(m, plan)


def test_solve_without_gpu_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    m, plan = _plan_cfg(0, 1.0)
    x = np.zeros(m.n)
    with pytest.raises(hb.HinesError) as e:
        plan.solve_host(x, x, x, x.copy())
    assert e.value.status == 4 and "no CPU fallback" in str(e.value)
