"""Test-side interpreter of the plan's policy tables (pure Python, fp64).

Executes exactly what the tables tell the resident kernel to do -- condense every segment (P1),
level-synchronous sweeps over the reduced tree with the pull hand-off (P2), expand (P3) -- one
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
            assert ka == 1 and kb == 2 and (int(A[1]) & ~(3 << 24)) == (int(B[1]) & ~(3 << 24)) and A[2] == B[2]
            mt, mb, hasq = int(A[1]) & 0xfff, (int(A[1]) >> 12) & 0xfff, (int(A[1]) >> 26) & 1
            mm = mt + mb + hasq
            assert B[0] == A[0] + mm - 1 and (hasq or (mt == 0 and mb == 0)) and abs(mt - mb) <= 1
            yield int(A[0]), mt, mb, hasq, int(A[2]), int(A[3])


def solve_with_tables(plan, m, d, u, b):
    """x for every cell that sits in an on-chip work item (NaN elsewhere)."""
    x = np.full(m.n, np.nan)
    rng_ = plan.table("item_cell_range").reshape(-1, 2)
    desc_off = plan.table("item_desc_offsets")
    lvl_off = plan.table("item_level_offsets")
    lvl_begin = plan.table("item_level_begin")
    desc = plan.table("item_desc").reshape(-1, 4)
    pnode_all = plan.table("item_pnode")
    nnode = plan.table("item_nnode")
    node_off = plan.table("item_node_offsets")
    rounds = plan.table("item_rounds")
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
                    # lane B: lower half b-1..q+1 bottom-up, fill-in coupling to b
                    eb = su[bp]; pD = pB = pdd = pdb = 0.0
                    if mb > 0:
                        j = bp - 1
                        Db, Bb = sd[j], sb[j]
                        for s_ in range(mb):
                            un = su[j]
                            dn, bn = (sd[j - 1], sb[j - 1]) if s_ + 1 < mb else (0.0, 0.0)
                            r = 1.0 / Db
                            g, h, c = un * r, eb * r, Bb * r
                            sd[j], su[j], sb[j] = g, h, c
                            pdd += h * eb; pdb += h * Bb
                            Db, Bb, eb = dn - g * un, bn - g * Bb, -h * un
                            j -= 1
                        pD, pB = Db, Bb
                    Dq, Bq = D + pD, B + pB
                    r = 1.0 / Dq
                    gq, hq = eb * r, ee * r
                    sd[q], su[q], sb[q] = gq, hq, Bq * r
                    ddt += hq * ee; dbt += hq * Bq
                    pdd += gq * eb; pdb += gq * Bq
                    rec = (sd[bp] - pdd, sb[bp] - pdb, -hq * eb, ddt, dbt)
                else:
                    rec = (D, B, ee, 0.0, 0.0)
                assert np.isnan(rD[node]), "node written twice"
                rD[node], rB[node], rU[node], pd[node], pb[node] = rec
            work.append((g0, g1, sd, su, sb, sg))
        # P2
        dsc = desc[desc_off[it]:desc_off[it + 1]]
        pn = pnode_all[node_off[it]:node_off[it + 1]]
        assert len(pn) == NN
        lb = lvl_begin[lvl_off[it]:lvl_off[it + 1]]
        nlev = len(lb) - 1
        for lev in range(nlev - 1, -1, -1):
            dd = np.zeros(lb[lev + 1] - lb[lev]); db = dd.copy()
            for e in range(lb[lev], lb[lev + 1]):
                w0, rest, cfirst, w3 = (int(v) for v in dsc[e])
                nseg, nlead = w0 & 0xffff, w3 & 0xffff
                if nseg == 0:
                    continue
                node = rest + nseg - 2 if nseg > 1 else e
                D, B = rD[node], rB[node]
                for c in range(nlead):
                    D -= pd[cfirst + c]; B -= pb[cfirst + c]
                for k in range(nseg):
                    r = 1.0 / D
                    U = rU[node]
                    f = U * r
                    rD[node], rB[node] = f, B * r
                    dde, dbe = f * U + pd[node], f * B + pb[node]
                    if k + 1 < nseg:
                        node = e if k + 2 == nseg else node - 1
                        D, B = rD[node] - dde, rB[node] - dbe
                dd[e - lb[lev]], db[e - lb[lev]] = dde, dbe
            # shuffle stage: lane e absorbs the nafter lanes to its right (same 32-lane tile)
            for e in range(lb[lev], lb[lev + 1]):
                w0 = int(dsc[e, 0])
                nseg, nafter = w0 & 0xffff, (w0 >> 16) & 0xff
                if nseg == 0:
                    continue
                j = e - lb[lev]
                assert j % 32 + nafter < 32, "sibling group leaves its tile"
                pd[e] = dd[j] + sum(dd[j + 1:j + 1 + nafter]); pb[e] = db[j] + sum(db[j + 1:j + 1 + nafter])
        # forward sweep by pointer jumping: x_v = c_v + g_v x_p(v), g = -f (a root: g = 0, p = itself)
        real = ~np.isnan(rD)
        g = np.where(real, -rD, 0.0); c = np.where(real, rB, 0.0); par = pn.astype(np.int64).copy()
        assert (par[~real] == np.nonzero(~real)[0]).all() and real[par[real]].all()
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
                xn = xq
                for j in range(q + 1, bp):
                    xn = (sb[j] - su[j] * xb) - sd[j] * xn
                    sb[j] = xn
            x[g0:g1] = sb
    return x
