"""Test-side interpreter of the plan's policy tables (pure Python, fp64).

Executes exactly what the tables tell the resident kernel to do -- condense every segment (P1),
the backward sweep over the reduced tree (tiers of warp groups in lock-step over the height, shuffle and
pull hand-off) and the pointer-jumping forward sweep (P2), expand (P3) -- one
"lane" at a time, so that a wrong table (a missing segment, a wrong node id, a child group the parent
does not pull) shows up on the CPU box as a wrong solution, before any GPU run.  It shares no code
with the library: it only reads tables through hines_plan_get_table.
"""
from __future__ import annotations

import numpy as np


def pairs(sg):
    """Segments of a chunk's lane list: groups of 32 lanes = 16 A lanes + their 16 B partners.
    Yields (a, mt, mb, hasq, node, tnode) per segment and checks the pairing."""
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
            mm = mt + mb + hasq
            assert (B[0] == A[0] + mt + 1 or not hasq) and (hasq or (mt == 0 and mb == 0)) and abs(mt - mb) <= 5
            yield int(A[0]), mt, mb, hasq, int(A[2]), int(A[3])


def parse_tasks(blob):
    """Per tier: (tier, [(lane_begin[33], steps, shuffle counts per step, turn-around lane mask)], entries, pull list, raw bytes)."""
    ntier = int(blob[0])
    tb = blob[1:2 + ntier]
    grp_off = -(-(2 + ntier) // 4) * 4
    ngroups = int(tb[-1])
    ent_off = grp_off + 36 * ngroups
    nent = int(blob[grp_off + 36 * (ngroups - 1) + 32]) if ngroups else 0
    ents = blob[ent_off:ent_off + 4 * nent].reshape(-1, 4)
    pull_off = ent_off + 4 * nent
    npull = int((ents[:, 3] & 0xffff).sum()) if nent else 0
    pull = blob[pull_off:pull_off + npull]
    raw = blob.view(np.uint8)
    out = []
    for t in range(ntier):
        groups = []
        for g in range(int(tb[t]), int(tb[t + 1])):
            gh = blob[grp_off + 36 * g:grp_off + 36 * g + 36]
            nsteps, boff = int(gh[33]), int(gh[34])
            groups.append((gh[:33], nsteps, raw[boff:boff + nsteps], int(gh[35]) & 0xffffffff))
        out.append((t, groups, ents, pull, raw))
    return out


def solve_with_tables(plan, m, d, u, b):
    """x for every cell that sits in an on-chip work item (NaN elsewhere)."""
    x = np.full(m.n, np.nan)
    rng_ = plan.table("item_cell_range").reshape(-1, 2)
    pnode_all = plan.table("item_pnode")
    nnode = plan.table("item_nnode")
    node_off = plan.table("item_node_offsets")
    rounds = plan.table("item_rounds")
    task_off = plan.table("item_task_offsets")
    task_blob = plan.table("item_task_blob")
    ch_off = plan.table("item_chunk_offsets")
    ch_rng = plan.table("chunk_comp_range").reshape(-1, 2)
    seg_off = plan.table("chunk_seg_offsets")
    segs = plan.table("chunk_seg").reshape(-1, 4)
    for it in range(len(rng_)):
        NN = int(nnode[it])
        rD = np.full(NN, np.nan); rB = rD.copy(); rU = rD.copy(); pd = rD.copy(); pb = rD.copy()
        work = []
        # P1
        for ch in range(ch_off[it], ch_off[it + 1]):
            g0, g1 = ch_rng[ch]
            sd = d[g0:g1].astype(np.float64).copy(); su = u[g0:g1].astype(np.float64).copy(); sb = b[g0:g1].astype(np.float64).copy()
            sg = segs[seg_off[ch]:seg_off[ch + 1]]
            assert len(sg) % 32 == 0
            for a, mt, mb, hasq, node, tnode in pairs(sg):
                # lane A: upper half a..q-1 top-down, fill-in coupling to t
                i = a
                D, B = sd[i], sb[i]
                ee = su[i] if tnode >= 0 else 0.0
                ddt = dbt = 0.0
                for _ in range(mt):
                    un, dn, bn = su[i + 1], sd[i + 1], sb[i + 1]
                    r = 1.0 / D
                    g, h, c = un * r, ee * r, B * r
                    sd[i], su[i], sb[i] = g, h, c
                    ddt += h * ee; dbt += h * B
                    D, B, ee = dn - g * un, bn - g * B, -h * un
                    i += 1
                if hasq:
                    q = a + mt; bp = q + 1 + mb
                    # lane B: q+1..b-1 top-down, fill-in coupling to q; arrives at b
                    j = q + 1
                    Db, Bb, eb = sd[j], sb[j], su[j]
                    pdd = pdb = 0.0
                    for _ in range(mb):
                        un, dn, bn = su[j + 1], sd[j + 1], sb[j + 1]
                        r = 1.0 / Db
                        g, h, c = un * r, eb * r, Bb * r
                        sd[j], su[j], sb[j] = g, h, c
                        pdd += h * eb; pdb += h * Bb
                        Db, Bb, eb = dn - g * un, bn - g * Bb, -h * un
                        j += 1
                    assert j == bp
                    Dq, Bq = D - pdd, B - pdb
                    r = 1.0 / Dq
                    gq, hq = eb * r, ee * r
                    sd[q], su[q], sb[q] = gq, hq, Bq * r
                    ddt += hq * ee; dbt += hq * Bq
                    rec = (Db - gq * eb, Bb - gq * Bq, -hq * eb, ddt, dbt)
                else:
                    rec = (D, B, ee, 0.0, 0.0)
                assert np.isnan(rD[node]), "node written twice"
                rD[node], rB[node], rU[node], pd[node], pb[node] = rec
            work.append((g0, g1, sd, su, sb, sg))
        # P2 backward: tiers of warp groups, lock-step over the height, a node in the lane of its first child
        pn = pnode_all[node_off[it]:node_off[it + 1]]
        assert len(pn) == NN
        blob = task_blob[task_off[it]:task_off[it + 1]]
        done = np.zeros(NN, bool)
        final = np.zeros(NN, bool)
        tiers = parse_tasks(blob)
        any_turn = any(g_[3] for t_ in tiers for g_ in t_[1])      # all root chains of an item turn around, or none
        for tier, groups, ents, pull, nshb in tiers:
            for gh, nsteps, nsh, turn in groups:
                outd = np.zeros(32); outb = np.zeros(32)
                pos = [int(gh[l]) for l in range(32)]
                for h in range(nsteps):
                    newd, newb = outd.copy(), outb.copy()
                    for lane in range(32):
                        first = True
                        while pos[lane] < gh[lane + 1]:
                            w0, mask, p0, w3 = (int(v) for v in ents[pos[lane]])
                            node, step = w0 & 0xfffff, (w0 >> 20) & 0xfff
                            pcount, run = w3 & 0xffff, w3 >> 16
                            # the run the kernel walks in its tight loop: entries right behind, same step, nothing to pull
                            assert pos[lane] + run < gh[lane + 1] or run == 0
                            for k in range(1, run + 1):
                                wk = [int(v) for v in ents[pos[lane] + k]]
                                assert (wk[0] >> 20) & 0xfff == step and wk[1] == 0 and wk[3] & 0xffff == 0 and wk[3] >> 16 == run - k
                            if step != h:
                                assert step > h
                                break
                            if first:
                                sd_, sb_ = outd[lane], outb[lane]
                                srcs = [l2 for l2 in range(32) if (mask >> l2) & 1]
                                assert len(srcs) <= nsh[h] and lane not in srcs
                                for l2 in srcs:
                                    sd_ += outd[l2]; sb_ += outb[l2]
                            else:                           # continuation of a run: only child = the node just computed
                                assert mask == 0
                                sd_, sb_ = newd[lane], newb[lane]
                            for c in pull[p0:p0 + pcount]:
                                assert done[c]
                                sd_ += pd[c]; sb_ += pb[c]
                            D, B = rD[node] - sd_, rB[node] - sb_
                            r = 1.0 / D
                            f = rU[node] * r
                            rD[node], rB[node] = f, B * r
                            newd[lane], newb[lane] = f * rU[node] + pd[node], f * B + pb[node]
                            assert not done[node]
                            done[node] = True
                            pos[lane] += 1
                            first = False
                            if pos[lane] >= gh[lane + 1]:
                                pd[node], pb[node] = newd[lane], newb[lane]       # hand-off slot
                    outd, outb = newd, newb
                assert all(pos[l] == gh[l + 1] for l in range(32))
                # a chain that ended in a root turns around: x_root = c_root, x = c - f x_parent down the lane's chain
                for l in range(32):
                    b_, e_ = int(gh[l]), int(gh[l + 1])
                    if (turn >> l) & 1:
                        assert e_ > b_ and rU[e_ - 1] == 0, "turn-around lane does not end in a root"
                        xv = rB[e_ - 1]
                        rD[e_ - 1] = 0.0
                        final[e_ - 1] = True
                        for k in range(e_ - 2, b_ - 1, -1):
                            xv = rB[k] - rD[k] * xv
                            rD[k], rB[k] = 0.0, xv
                            final[k] = True
                    elif e_ > b_ and any_turn:
                        assert pn[e_ - 1] != e_ - 1, "a chain that ends in a root must turn around"
        assert done.all()
        # forward sweep by pointer jumping: x_v = c_v + g_v x_p(v), g = -f (a root: g = 0, p = itself)
        real = ~np.isnan(rD)
        g = np.where(real, -rD, 0.0); c = np.where(real, rB, 0.0); par = pn.astype(np.int64).copy()
        assert (par[~real] == np.nonzero(~real)[0]).all() and real[par[real]].all()
        assert (par[final] == np.nonzero(final)[0]).all(), "a final node reads itself"
        for _ in range(int(rounds[it])):
            g, c, par = g * g[par], c + g * c[par], par[par]
        assert (g[real] == 0).all(), "not enough pointer-jumping rounds"
        rB = c
        # P3
        for g0, g1, sd, su, sb, sg in work:
            for a, mt, mb, hasq, node, tnode in pairs(sg):
                xb = rB[node]
                xt = rB[tnode] if tnode >= 0 else 0.0
                if not hasq:
                    sb[a] = xb
                    continue
                q = a + mt; bp = q + 1 + mb
                xq = (sb[q] - su[q] * xt) - sd[q] * xb
                sb[q] = xq; sb[bp] = xb
                xn = xq
                for j in range(q - 1, a - 1, -1):
                    xn = (sb[j] - su[j] * xt) - sd[j] * xn
                    sb[j] = xn
                xn = xb
                for j in range(bp - 1, q, -1):
                    xn = (sb[j] - su[j] * xq) - sd[j] * xn
                    sb[j] = xn
            x[g0:g1] = sb
    return x
