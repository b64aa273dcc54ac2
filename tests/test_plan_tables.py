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
from plan_interpreter import pairs, parse_tasks

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
    assert ctypes.sizeof(hb.Options) == 36 and ctypes.sizeof(hb.PlanInfo) == 152


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


def _check_policy(m, plan, max_segment=0):
    """Validity invariants (policy-free): every cell in exactly one on-chip item or on the streaming
    path; the chunks of an item tile its compartment range; segments tile every branch exactly, each
    inside one chunk and listed once; node ids are unique; a segment's upper node is the node of the
    compartment above it; every branch has one lane on its level; sibling groups of at most 32 sit in
    one 32-lane tile and their first lane absorbs the others, larger groups are pulled one by one;
    shared-memory need within the class; launch order a permutation."""
    T = oracle.tables(m.parent, m.cell_offsets)
    w = 8 if plan.dtype == hb.F64 else 4
    E = 16 // w
    cell_item = plan.table("cell_item")
    rng_ = plan.table("item_cell_range").reshape(-1, 2)
    pnode = plan.table("item_pnode")
    nnode = plan.table("item_nnode")
    node_off = plan.table("item_node_offsets")
    rounds = plan.table("item_rounds")
    ch_off = plan.table("item_chunk_offsets")
    ch_rng = plan.table("chunk_comp_range").reshape(-1, 2)
    seg_off = plan.table("chunk_seg_offsets")
    segs = plan.table("chunk_seg").reshape(-1, 4)
    cls = plan.table("item_class")
    cls_smem = plan.table("class_smem_bytes")
    cls_cluster = plan.table("class_cluster")
    cls_threads = plan.table("class_threads")
    order = plan.table("item_launch_order")
    nitems = len(cls)
    assert sorted(order.tolist()) == list(range(nitems))
    assert (np.diff(cls[order]) >= 0).all()
    assert ((cls_threads % 32 == 0) & (cls_threads >= 32) & (cls_threads <= 1024)).all()
    info = plan.info
    assert info.n_resident_items == nitems and info.n_chunks == len(ch_rng)
    seen_cells = np.zeros(m.ncells, bool)
    useful = 0
    nsep_total = 0
    for it in range(nitems):
        c0, c1 = rng_[it]
        assert c1 > c0 and (cell_item[c0:c1] == it).all()
        seen_cells[c0:c1] = True
        comp0 = m.cell_offsets[c0]; n_it = m.cell_offsets[c1] - comp0
        nch = ch_off[it + 1] - ch_off[it]
        assert nch == cls_cluster[cls[it]] and (nch == 1 or c1 - c0 == 1)
        cr = ch_rng[ch_off[it]:ch_off[it + 1]]
        assert cr[0, 0] == comp0 and cr[-1, 1] == comp0 + n_it and (cr[1:, 0] == cr[:-1, 1]).all()
        pn_sweep = pnode[node_off[it]:node_off[it + 1]]
        # ITEM_PNODE is the parent the FORWARD sweep reads: a node of a lane chain that ends in a root is final
        # after the backward sweep's turn-around and reads itself.  pn = the parent in the reduced tree: for those
        # nodes the next entry of the lane's chain (node id = entry index).
        pn = pn_sweep.copy()
        blob_ = plan.table("item_task_blob")[plan.table("item_task_offsets")[it]:plan.table("item_task_offsets")[it + 1]]
        tiers_ = parse_tasks(blob_)
        any_turn = any(g_[3] for t_ in tiers_ for g_ in t_[1])     # all root chains of an item turn around, or none
        for _t, groups_, _e, _p, _r in tiers_:
            for gh_, _ns, _nsh, turn_ in groups_:
                for l_ in range(32):
                    b_, e_ = int(gh_[l_]), int(gh_[l_ + 1])
                    if (turn_ >> l_) & 1:
                        assert e_ > b_ and (pn_sweep[b_:e_] == np.arange(b_, e_)).all()
                        pn[b_:e_ - 1] = np.arange(b_ + 1, e_)
                    elif e_ > b_ and any_turn:
                        assert pn_sweep[e_ - 1] != e_ - 1          # a chain that ends in a root turns around
        assert len(pn) == nnode[it]
        # segments of all chunks -> node of every separator compartment (item-local position)
        node_at = {}                     # separator position -> node
        seg_of_node = {}
        covered = np.zeros(n_it, int)
        nlanes_max = 0
        # segment target of the item: the option, or by default 40 in a block of its own, 64 in a cluster
        S_it = max_segment if max_segment else (40 if ch_off[it + 1] - ch_off[it] == 1 else 64)
        for r, ch in enumerate(range(ch_off[it], ch_off[it + 1])):
            sg = segs[seg_off[ch]:seg_off[ch + 1]]
            nlanes_max = max(nlanes_max, len(sg))
            base = cr[r, 0] - comp0
            for a, mt_, mb_, hasq_, node, tnode in pairs(sg):
                mm = mt_ + mb_ + hasq_
                assert 0 <= node < nnode[it] and node not in seg_of_node
                assert 0 <= a and a + mm < cr[r, 1] - cr[r, 0] and 0 <= mm < 2 * S_it
                seg_of_node[int(node)] = (int(base + a), int(mm), int(tnode))
                node_at[int(base + a + mm)] = int(node)
                covered[base + a:base + a + mm + 1] += 1
                useful += int(mm)
            L = -(-(cr[r, 0] % E + cr[r, 1] - cr[r, 0]) // E) * E
            tb = plan.table("item_task_offsets")
            meta = int(tb[it + 1] - tb[it]) + -(-nnode[it] // 4) * 4
            need = 16 + 3 * L * w + 16 * len(sg) + (6 * (-(-nnode[it] // E) * E) * w + 4 * meta if r == 0 else 0)
            assert need <= cls_smem[cls[it]] <= 232448
        assert (covered == 1).all()
        nsep_total += len(seg_of_node)
        # branches: one lane each, on its level; node chain from the top: e, rest, rest+1, ...
        want = {}
        for c in range(c0, c1):
            sh = m.cell_offsets[c] - comp0
            for j in range(T.cell_branch_offsets[c], T.cell_branch_offsets[c + 1]):
                pc = T.branch_parent_comp[j]
                want[int(T.branch_start[j] + sh)] = (int(T.branch_len[j]), -1 if pc < 0 else int(pc + sh), int(T.branch_level[j]))
        seg_at = {a: (mm, node, t) for node, (a, mm, t) in seg_of_node.items()}       # by first compartment
        lanes_seen = set()
        for start, (ln, pc, lw) in want.items():
            nseg = max(1, (5 * ln + 2 * S_it) // (5 * S_it))       # len / max_segment + 0.4, cut off
            sj = -(-ln // nseg)
            if nseg > 1 and sj % 2 == 0:
                sj += 1                                      # odd: the segments of a branch start on distinct banks
            nseg = -(-ln // sj)                              # no empty segment
            end = start + ln - 1
            prev = node_at[pc] if pc >= 0 else -1
            for k in range(nseg):                            # k-th segment from the top
                q = nseg - 1 - k
                b_ = end - q * sj
                a_ = max(start, b_ - sj + 1)
                mm, node, tn = seg_at[a_]
                assert mm == b_ - a_ and tn == prev, (it, start, k)
                assert pn[node] == (prev if prev >= 0 else node)             # a root reads itself (its f is 0)
                prev = node
            lanes_seen.add(start)
        assert len(lanes_seen) == len(want) and len(seg_of_node) == nnode[it]
        # backward-sweep tasks: every node once; a node's step is above its children's; children of the same
        # tier sit in the same group: the first in the node's own lane, the others in its lane mask; children
        # of earlier tiers are in its pull list; at most 32 lanes per group
        blob = plan.table("item_task_blob")[plan.table("item_task_offsets")[it]:plan.table("item_task_offsets")[it + 1]]
        where = {}
        for tier, groups, ents, pull, raw in parse_tasks(blob):
            for gi, (gh, nsteps, nsh, _turn) in enumerate(groups):
                for lane in range(32):
                    prev = None
                    for k in range(int(gh[lane]), int(gh[lane + 1])):
                        node, step = int(ents[k, 0]) & 0xfffff, (int(ents[k, 0]) >> 20) & 0xfff
                        assert node not in where and step < nsteps
                        where[node] = (tier, gi, lane, step, k)
                        if prev is not None:                 # the lane's chain: each node the parent of the one before
                            assert pn[prev[0]] == node and step >= prev[1]
                        prev = (node, step)
        assert sorted(where) == list(range(nnode[it]))
        kids_of = {}
        for v in range(nnode[it]):
            if pn[v] != v:
                kids_of.setdefault(int(pn[v]), []).append(v)
        _, _, ents, pull, _ = parse_tasks(blob)[0]
        for v, (tier, gi, lane, step, k) in where.items():
            same = [c for c in kids_of.get(v, []) if where[c][0] == tier]
            lower = [c for c in kids_of.get(v, []) if where[c][0] != tier]
            assert all(where[c][0] < tier for c in lower)
            assert sorted(int(c) for c in pull[int(ents[k, 2]):int(ents[k, 2]) + (int(ents[k, 3]) & 0xffff)]) == sorted(lower)
            mask = int(ents[k, 1]) & 0xffffffff
            if same:
                assert all(where[c][1] == gi for c in same)
                if where[same[0]][3] == step:                # a run (plain chains only): the single child's step
                    assert len(same) == 1 and mask == 0
                else:
                    assert all(where[c][3] < step for c in same)
                assert where[min(same)][2] == lane
                assert mask == sum(1 << where[c][2] for c in same if c != min(same))
            else:
                assert mask == 0 and (lower or step == 0)
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
    (2, 0.003, dict(max_segment=2)), (3, 0.002, dict(max_segment=16)),
    (2, 0.004, dict(chunk_smem_bytes=30000, cluster_max=16)), (1, 0.002, dict(max_segment=5, chunk_smem_bytes=8000)),
    (3, 0.002, dict(chunk_smem_bytes=40000, cluster_max=4)),
])
def test_policy_tables_valid(cfg, scale, kw):
    m, plan = _plan_cfg(cfg, scale, **kw)
    _check_policy(m, plan, kw.get("max_segment", 0))
    _check_interpreted(m, plan)


def test_policy_star_with_many_siblings_and_odd_offsets():
    star = np.array([-1] + [0] * 70, np.int32)                        # 70 siblings: more than a tile -> pulled one by one
    ps = [star, random_parent(33, 1), np.array([-1], np.int32), random_parent(200, 2, .7), star[:40],
          random_parent(1001, 3, .97)]
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    m = mg.Morphology(np.concatenate(ps), offs)
    for kw in ({}, dict(dtype=hb.F32), dict(policy_flags=hb.POLICY_NO_GROUPING), dict(max_segment=3),
               dict(chunk_smem_bytes=6000, max_segment=4)):
        plan = hb.Plan(m.parent, m.cell_offsets, **kw)
        _check_policy(m, plan, kw.get("max_segment", 0))
        _check_interpreted(m, plan)
        blob = plan.table("item_task_blob")[:plan.table("item_task_offsets")[1]]
        assert any(int(e[3]) == 70 for t in parse_tasks(blob)[:1] for e in t[2])      # the star's root pulls its 70 children


def test_clusters_take_the_cells_too_large_for_one_block():
    m, plan = _plan_cfg(3, 0.004)
    info = plan.info
    assert info.n_cluster_cells > 0 and info.n_stream_cells == 0
    cl = plan.table("class_cluster")
    assert cl.min() == 1 and cl.max() <= 16 and (np.diff(cl) <= 0).all()
    m, plan = _plan_cfg(3, 0.004, policy_flags=hb.POLICY_POW2_CLUSTERS)
    assert set(plan.table("class_cluster").tolist()) <= {1, 2, 4, 8, 16}
    m, plan = _plan_cfg(3, 0.004, policy_flags=hb.POLICY_NO_CLUSTER)
    assert plan.info.n_cluster_cells == 0 and (plan.table("class_cluster") == 1).all()


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
