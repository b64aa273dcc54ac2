"""Test-side interpreter of the plan's policy tables (pure Python, fp64).

Executes exactly what the tables tell the resident kernel to do -- condense every segment (P1),
level-synchronous sweeps over the reduced tree with the pull hand-off (P2), expand (P3) -- one
"lane" at a time, so that a wrong table (a missing segment, a wrong node id, a child group the parent
does not pull) shows up on the CPU box as a wrong solution, before any GPU run.  It shares no code
with the library: it only reads tables through hines_plan_get_table.
"""
from __future__ import annotations

import numpy as np


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
            for a, mm, node, tnode in sg:
                if node < 0:
                    continue
                i = a
                D, B = sd[i], sb[i]
                ee = su[i] if tnode >= 0 else 0.0
                ddt = dbt = 0.0
                for _ in range(mm):
                    un, dn, bn = su[i + 1], sd[i + 1], sb[i + 1]
                    r = 1.0 / D
                    g, h, c = un * r, ee * r, B * r
                    sd[i], su[i], sb[i] = g, h, c
                    ddt += h * ee; dbt += h * B
                    D, B, ee = dn - g * un, bn - g * B, -h * un
                    i += 1
                assert np.isnan(rD[node]), "node written twice"
                rD[node], rB[node], rU[node], pd[node], pb[node] = D, B, ee, ddt, dbt
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
            for a, mm, node, tnode in sg:
                if node < 0:
                    continue
                xn = rB[node]
                xt = rB[tnode] if tnode >= 0 else 0.0
                sb[a + mm] = xn
                for j in range(mm - 1, -1, -1):
                    xn = (sb[a + j] - su[a + j] * xt) - sd[a + j] * xn
                    sb[a + j] = xn
            x[g0:g1] = sb
    return x
