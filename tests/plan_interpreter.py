"""Test-side interpreter of the plan's policy tables (pure Python, fp64).

Executes exactly what the tables tell the resident kernel to do -- stage the runs of every part, condense
every segment (P1), the level-synchronous backward sweep over the part's reduced forest with the pull
hand-off (P2), the exchange between the parts of one cell (exports -> ghost children, parent's x -> ghost
parents), the pointer-jumping forward sweep, expand (P3), store run by run -- one "lane" at a time, so
that a wrong table (a missing segment, a wrong node id, a child the parent does not pull, a wrong run)
shows up on the CPU box as a wrong solution, before any GPU run.  It shares no code with the library: it
only reads tables through hines_plan_get_table.
"""
from __future__ import annotations

import numpy as np

HDR = {"meta_off": 0, "meta_len": 2, "run_off": 3, "nrun": 4, "tx_elems": 5, "L": 6, "n": 7, "nnode": 8,
       "nlevnode": 9, "nlev": 10, "rounds": 11, "kp_off": 12, "exp_off": 13, "gh_off": 14, "seg_off": 15,
       "nexp": 16, "nghost": 17, "nseg_lanes": 18, "xch_base": 19, "xs0": 20, "item": 21, "rank": 22, "flags": 23, "ntoplev": 24, "lowlev": 25, "maxwidth": 26}


class Part:
    """One part's tables, parsed from PART_HEADER / PART_META / PART_RUNS."""

    def __init__(self, hdr, meta_all, runs_all):
        h = {k: int(hdr[i]) for k, i in HDR.items()}
        h["meta_off"] = int(hdr[0:2].view(np.int64)[0])
        self.h = h
        meta = meta_all[h["meta_off"]:h["meta_off"] + h["meta_len"]]
        self.lb = meta[:h["nlev"] + 1]
        kp4 = meta[h["kp_off"]:h["kp_off"] + 4 * h["nnode"]].reshape(-1, 4)
        self.kp4 = kp4
        info = kp4[:, 2]
        self.ghost = info < 0
        self.top = np.where(self.ghost, 0, (info >> 29) & 1)   # an ancestor of a ghost child
        self.nc = np.where(self.ghost, 0, info & 0xfff)
        self.pnode = kp4[:, 3]
        self.chains = bool(h["flags"] & 1)
        self.factored = bool(h["flags"] & 2)
        self.exps = meta[h["exp_off"]:h["exp_off"] + 4 * h["nexp"]].reshape(-1, 4)
        self.ghosts = meta[h["gh_off"]:h["gh_off"] + 4 * h["nghost"]].reshape(-1, 4)
        self.seg = meta[h["seg_off"]:h["seg_off"] + 4 * h["nseg_lanes"]].reshape(-1, 4)
        assert h["seg_off"] + 4 * h["nseg_lanes"] == h["meta_len"] and h["meta_len"] % 4 == 0
        assert all(h[k] % 4 == 0 for k in ("kp_off", "exp_off", "gh_off", "seg_off"))
        self.runs = runs_all[h["run_off"]:h["run_off"] + h["nrun"]]
        assert int(self.lb[-1]) == h["nlevnode"] and h["nnode"] == h["nlevnode"] + h["nexp"]

    def children(self, v, w):
        """Node ids of v's children from the byte offsets of their hand-off slots (record = 6 values of w bytes,
        slot at value 4; the all-zero record sits at index nnode); children beyond the second are consecutive."""
        nc = int(self.nc[v])
        ids = []
        for q in range(2):
            off = int(self.kp4[v, q])
            assert (off - 4 * w) % (6 * w) == 0
            idx = (off - 4 * w) // (6 * w)
            if q < nc:
                ids.append(idx)
            else:
                assert idx == self.h["nnode"], "absent child points at the zero record"
        ids += [ids[1] + k for k in range(1, nc - 1)]
        return ids


def pairs(sg):
    """Segments of a part's lane list: groups of 32 lanes = 16 A lanes + their 16 B partners.
    Yields (a, mt, mb, hasq, node, tnode) per segment and checks the pairing."""
    assert len(sg) % 32 == 0
    for g in range(0, len(sg), 32):
        for k in range(16):
            A, B = sg[g + k], sg[g + 16 + k]
            ka, kb = (int(A[1]) >> 24) & 3, (int(B[1]) >> 24) & 3
            if ka == 0:
                assert kb == 0 and A[2] == -1 and B[2] == -1
                continue
            msk = ~((3 << 24) | (15 << 27))                # kind and the lane's start delay differ between A and B
            assert ka == 1 and kb == 2 and (int(A[1]) & msk) == (int(B[1]) & msk) and A[2] == B[2]
            mt, mb, hasq = int(A[1]) & 0xfff, (int(A[1]) >> 12) & 0xfff, (int(A[1]) >> 26) & 1
            assert (B[0] == A[0] + mt + 1 or not hasq) and (hasq or (mt == 0 and mb == 0)) and abs(mt - mb) <= 5
            yield int(A[0]), mt, mb, hasq, int(A[2]), int(A[3])


def segments(sg):
    """Segments of a part's lane list, two-lane and four-lane groups alike: yields (a, lens, node, tnode) where lens are
    the steps of the segment's lanes (its halves / quarters; [] for a segment that is its separator alone) and the
    middle nodes sit between them: the segment covers a .. a + sum(lens) + len(lens) - 1, the last one its separator."""
    assert len(sg) % 32 == 0
    for g in range(0, len(sg), 32):
        kinds = [(int(sg[g + l][1]) >> 24) & 3 for l in range(32)]
        if 3 in kinds:                                     # a four-lane group: lane k + 8 j = quarter j of segment k
            assert all(k in (0, 3) for k in kinds)
            for k in range(8):
                Ls = [sg[g + k + 8 * j] for j in range(4)]
                if kinds[k] == 0:
                    assert all(kinds[k + 8 * j] == 0 and Ls[j][2] == -1 for j in range(4))
                    continue
                lens, pos = [], int(Ls[0][0])
                for j in range(4):
                    w = int(Ls[j][1])
                    assert kinds[k + 8 * j] == 3 and (w >> 12) & 3 == j and (w >> 26) & 1 == 1
                    assert int(Ls[j][0]) == pos and Ls[j][2] == Ls[0][2] and (j == 0 or Ls[j][3] == -1)
                    lens.append(w & 0xfff)
                    pos += lens[-1] + 1
                # a quarter boundary moves by at most two nodes: a quarter is within 4 of the balanced length
                assert max(lens) - min(lens) <= 9 and min(lens) >= 1
                yield int(Ls[0][0]), lens, int(Ls[0][2]), int(Ls[0][3])
        else:
            for a, mt, mb, hasq, node, tnode in pairs(sg[g:g + 32]):
                yield a, ([mt, mb] if hasq else []), node, tnode


def parts_of(plan):
    hdrs = plan.table("part_header").reshape(-1, 32)
    meta = plan.table("part_meta")
    runs = plan.table("part_runs").reshape(-1, 4)
    return [Part(h, meta, runs) for h in hdrs]


class _PartState:
    def __init__(self, part, d, u, b, n_total, E):
        h = part.h
        self.p = part
        L = h["L"]
        self.sd = np.full(L, np.nan); self.su = np.full(L, np.nan); self.sb = np.full(L, np.nan)
        tx = 0
        cursor = 0
        for g, ln, so, wd in part.runs:
            g, ln, so, wd = int(g), int(ln), int(so), int(wd)
            assert ln > 0 and so % E == g % E and so >= cursor and so + ln <= L, "run staged at the parity of its global index"
            cursor = so + ln
            ga, ge = g - g % E, min(-(-(g + ln) // E) * E, n_total // E * E)
            tx += max(0, ge - ga)
            # word 3: what the loader and the store would otherwise compute per run
            head = min(ln, (E - g % E) % E)
            tail = max(head, (g + ln) // E * E - g)
            assert wd & 0xffff == max(0, ge - ga) and (wd >> 16) & 15 == head and (wd >> 20) & 15 == ln - tail
            assert (wd >> 24) == (1 if g + ln > ge else 0)
            self.sd[so:so + ln] = d[g:g + ln]; self.su[so:so + ln] = u[g:g + ln]; self.sb[so:so + ln] = b[g:g + ln]
        assert tx == h["tx_elems"] and L % E == 0 and sum(int(r[1]) for r in part.runs) == h["n"]
        nn = h["nnode"]
        self.rec = np.full((nn + 1, 6), np.nan)
        self.rec[nn, 4:6] = 0.0                             # the all-zero record
        self.w = 16 // E

    def condense(self):
        """P1: the lanes of a segment (two or four), all top-down with fill-in to the lane's top; then the middle nodes
        in turn, by the segment's first lane."""
        sd, su, sb, rec = self.sd, self.su, self.sb, self.rec
        for a, lens, node, tnode in segments(self.p.seg):
            if not lens:
                new = (sd[a], sb[a], -(su[a] if tnode >= 0 else 0.0), 0.0, 0.0)
            else:
                arr, start = [], a
                for j, mj in enumerate(lens):
                    i = start
                    D, B = sd[i], sb[i]
                    ee = su[i] if (j > 0 or tnode >= 0) else 0.0
                    ddt = dbt = 0.0
                    for _ in range(mj):
                        un, dn, bn = su[i + 1], sd[i + 1], sb[i + 1]
                        r = 1.0 / D
                        g, h, c = un * r, ee * r, B * r
                        sd[i], su[i], sb[i] = g, h, c
                        ddt += h * ee; dbt += h * B
                        D, B, ee = dn - g * un, bn - g * B, -h * un
                        i += 1
                    arr.append((D, B, ee, ddt, dbt))
                    start = i + 1
                Dc, Bc, et, ddt, dbt = arr[0]
                q = a + lens[0]
                for s_ in range(1, len(lens)):
                    pD, pB, pe, pdd, pdb = arr[s_]
                    Dq, Bq = Dc - pdd, Bc - pdb
                    r = 1.0 / Dq
                    gq, hq = pe * r, et * r
                    sd[q], su[q], sb[q] = gq, hq, Bq * r
                    ddt += hq * et; dbt += hq * Bq
                    Dc, Bc, et = pD - gq * pe, pB - gq * Bq, -hq * pe
                    q += lens[s_] + 1
                new = (Dc, Bc, -et, ddt, dbt)                   # slot 2 holds -U
            assert 0 <= node < self.p.h["nlevnode"] and np.isnan(rec[node, 0]), "node written twice"
            assert not self.p.ghost[node], "a ghost child has no segment"
            rec[node, 0], rec[node, 1], rec[node, 2], rec[node, 4], rec[node, 5] = new

    def cables(self):
        """A part of unbranched cables: lb[] = first node of each cable; the reduced chain of a cable is a
        tridiagonal system (the kernel solves it by cyclic reduction inside a warp; any exact solve is the same)."""
        p, rec = self.p, self.rec
        x = np.zeros(p.h["nnode"])
        for c in range(p.h["nlev"]):
            n0, n1 = int(p.lb[c]), int(p.lb[c + 1])
            m = n1 - n0
            assert 1 <= m <= 32
            A = np.zeros((m, m)); rhs = np.zeros(m)
            for i in range(m):
                A[i, i] = rec[n0 + i, 0] - (rec[n0 + i + 1, 4] if i + 1 < m else 0.0)
                rhs[i] = rec[n0 + i, 1] - (rec[n0 + i + 1, 5] if i + 1 < m else 0.0)
                if i > 0:
                    A[i, i - 1] = A[i - 1, i] = -rec[n0 + i, 2]
                    assert p.pnode[n0 + i] == n0 + i - 1
                else:
                    assert p.pnode[n0] == n0 and rec[n0, 2] == 0
            x[n0:n1] = np.linalg.solve(A, rhs)
        return x

    def backward(self, sweep):
        """P2 backward: deepest level first; a node pulls its children (first two by their slot offsets, the rest
        consecutive, ascending).  sweep 0: everything that does not wait for another part (levels nlev-1 .. lowlev,
        nodes that are not top nodes); sweep 1: the top nodes (levels ntoplev-1 .. 0), after the ghost children got
        their hand-off."""
        p, rec = self.p, self.rec
        if sweep == 0:
            self.done = np.zeros(p.h["nlevnode"], bool)
        done = self.done
        if sweep == 1:                                       # every ghost child has received its hand-off by now
            gc = np.nonzero(p.ghost[:p.h["nlevnode"]])[0]
            assert not np.isnan(rec[gc, 4]).any(), "ghost child without its hand-off"
            done[gc] = True
        lv = range(p.h["nlev"] - 1, p.h["lowlev"] - 1, -1) if sweep == 0 else range(p.h["ntoplev"] - 1, -1, -1)
        for l in lv:
            assert p.lb[l + 1] - p.lb[l] <= p.h["maxwidth"]
            for v in range(int(p.lb[l]), int(p.lb[l + 1])):
                if p.ghost[v] or p.top[v] != sweep:
                    continue
                D, B, Un = rec[v, 0], rec[v, 1], rec[v, 2]
                assert not np.isnan(D), "node without a segment"
                for c in p.children(v, self.w):
                    assert done[c] and p.lb[l + 1] <= c < p.lb[l + 2], "children sit on the next level"
                    assert p.pnode[c] == v or p.ghost[c]
                    D -= rec[c, 4]; B -= rec[c, 5]
                r = 1.0 / D
                g = Un * r
                rec[v, 0], rec[v, 1] = g, B * r
                rec[v, 4], rec[v, 5] = g * Un + rec[v, 4], rec[v, 5] - g * B
                assert not done[v]
                done[v] = True
        if sweep == 1:
            assert done.all()

    def forward_top(self):
        """x of the top nodes, level by level from the root; a finished node holds {g, c} = {0, x}."""
        p, rec = self.p, self.rec
        for l in range(p.h["ntoplev"]):
            for v in range(int(p.lb[l]), int(p.lb[l + 1])):
                if p.ghost[v] or not p.top[v]:
                    continue
                pn = int(p.pnode[v])
                xp = 0.0 if pn == v else rec[pn, 1]
                assert pn == v or (p.top[pn] and rec[pn, 0] == 0.0), "a top node's parent is a finished top node"
                rec[v, 0], rec[v, 1] = 0.0, rec[v, 1] + rec[v, 0] * xp

    def forward(self):
        """P2 forward by pointer jumping; returns x per node."""
        p, rec = self.p, self.rec
        nn = p.h["nnode"]
        par = p.pnode.astype(np.int64).copy()
        ghost_child = p.ghost
        g = np.where(ghost_child, 0.0, rec[:nn, 0]); c = np.where(ghost_child, 0.0, rec[:nn, 1])
        assert (par[ghost_child] == np.nonzero(ghost_child)[0]).all()
        assert (par[p.h["nlevnode"]:] == np.arange(p.h["nlevnode"], nn)).all(), "a ghost parent reads itself"
        assert not np.isnan(g[~ghost_child]).any() and not np.isnan(c[~ghost_child]).any()
        for _ in range(p.h["rounds"]):
            g, c, par = g * g[par], c + g * c[par], par[par]
        assert (g[~ghost_child] == 0).all(), "not enough pointer-jumping rounds"
        return c

    def expand(self, xnode, x, E):
        """P3 + the store, run by run."""
        sd, su, sb = self.sd, self.su, self.sb
        for a, lens, node, tnode in segments(self.p.seg):
            xb = xnode[node]
            xt = xnode[tnode] if tnode >= 0 else 0.0
            if not lens:
                sb[a] = xb
                continue
            qs = [a + lens[0]]
            for s_ in range(1, len(lens) - 1):
                qs.append(qs[-1] + lens[s_] + 1)
            bp = qs[-1] + lens[-1] + 1
            xq, xnext = {}, xb
            for s_ in range(len(qs) - 1, -1, -1):              # the middle nodes, from the separator upward
                q = qs[s_]
                xq[s_] = (sb[q] - su[q] * xt) - sd[q] * xnext
                sb[q] = xq[s_]
                xnext = xq[s_]
            sb[bp] = xb
            start = a
            for j, mj in enumerate(lens):
                xT = xt if j == 0 else xq[j - 1]
                xn = xq[j] if j < len(qs) else xb
                for i in range(start + mj - 1, start - 1, -1):
                    xn = (sb[i] - su[i] * xT) - sd[i] * xn
                    sb[i] = xn
                start += mj + 1
        for g, ln, so, _ in self.p.runs:
            assert np.isnan(x[g:g + ln]).all(), "compartment stored twice"
            x[g:g + ln] = sb[so:so + ln]


def solve_with_tables(plan, m, d, u, b):
    """x for every cell that sits in an on-chip work item (NaN elsewhere)."""
    x = np.full(m.n, np.nan)
    E = 2 if plan.np_dtype == np.float64 else 4
    d = np.asarray(d, np.float64); u = np.asarray(u, np.float64); b = np.asarray(b, np.float64)
    parts = parts_of(plan)
    poff = plan.table("item_part_offsets")
    kind = plan.table("item_kind")
    for it in range(len(kind)):
        ps = [_PartState(parts[k], d, u, b, m.n, E) for k in range(poff[it], poff[it + 1])]
        assert (kind[it] == 0) == (len(ps) == 1)
        for r, s in enumerate(ps):
            assert s.p.h["item"] == it and s.p.h["rank"] == r
            assert (r == 0 or s.p.h["nghost"] == 0) and (r > 0 or s.p.h["nexp"] == 0)
        if ps[0].p.chains:
            assert len(ps) == 1 and ps[0].p.h["rounds"] == 0
            ps[0].condense()
            ps[0].expand(ps[0].cables(), x, E)
            continue
        ps[0].condense(); ps[0].backward(0)              # part 0's own sub-trees do not wait for the others
        # sub-tree parts: condense, sweep backward, export the roots' hand-off values to part 0's ghost children
        exported = set()
        for s in ps[1:]:
            s.condense(); s.backward(0); s.backward(1)
            assert not s.p.top.any() and not s.p.chains
            for v, gp, gx, p0 in s.p.exps:                      # {node, ghost parent, ghost child / exchange slot, parent in part 0}
                if kind[it] == 1:
                    ghost = int(gx)
                else:                                            # split item: through exchange slot gx
                    hit = [int(g[0]) for g in ps[0].p.ghosts if g[1] == gx]
                    assert len(hit) == 1
                    ghost = hit[0]
                    p0 = int([g[2] for g in ps[0].p.ghosts if g[1] == gx][0])
                assert ps[0].p.ghost[ghost] and ghost not in exported
                exported.add(ghost)
                ps[0].rec[ghost, 4], ps[0].rec[ghost, 5] = s.rec[v, 4], s.rec[v, 5]
                # the ghost child's parent in part 0 is the node whose x the root reads back
                gl = [g for g in ps[0].p.ghosts if g[0] == ghost][0]
                assert int(gl[2]) == int(p0) and ps[0].p.top[int(p0)]
        assert len(exported) == ps[0].p.h["nghost"]
        ps[0].backward(1)
        ps[0].forward_top()
        xtop = ps[0].rec[:, 1].copy()                    # what the other parts read: x of the top nodes
        x0 = ps[0].forward()
        ps[0].expand(x0, x, E)
        landed = [dict() for _ in ps]
        if kind[it] == 1:
            # cluster item: rank 0 SENDS the parent's x into the block of the part that waits for it, behind the export's
            # entry: the ghost child's entry names {rank << 20 | 4-byte word from the start of that block's shared memory}
            w = 8 if E == 2 else 4
            for gc, _, p0, dest in ps[0].p.ghosts:
                r, word = int(dest) >> 20, int(dest) & 0xfffff
                assert 1 <= r < len(ps)
                h = ps[r].p.h
                NN = -(-(h["nnode"] + 1) // E) * E
                rel = word - (16 + 512 + 6 * w * NN) // 4 - h["exp_off"]
                assert rel >= 0 and rel % 4 == 2 and rel // 4 < h["nexp"] and rel // 4 not in landed[r]
                landed[r][rel // 4] = xtop[int(p0)]
        for r, s in enumerate(ps):
            if r == 0:
                continue
            for e, (v, gp, gx, p0) in enumerate(s.p.exps):
                if kind[it] != 1:
                    p0 = int([g[2] for g in ps[0].p.ghosts if g[1] == gx][0])
                    landed[r][e] = xtop[p0]
                assert gp >= s.p.h["nlevnode"] and s.p.pnode[v] == gp
                assert xtop[p0] == x0[p0] and landed[r][e] == xtop[p0]
                s.rec[gp, 0], s.rec[gp, 1] = 0.0, landed[r][e]
            s.expand(s.forward(), x, E)
    return x
