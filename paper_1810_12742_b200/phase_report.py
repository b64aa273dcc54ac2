"""Phase clocks per size class:  python -m paper_1810_12742_b200.phase_report [--config C ...] [--dtype f64|f32]

Solves one synthetic batch (morphgen config C) a few times, then once more with the plan's phase clocks on
(hines_plan_enable_phase_clocks, include/hines.h): thread 0 of every block stamps %globaltimer at block start, inputs
landed, P1 done, backward sweep done, exchange + forward sweep done, P3 done, x stored.  Prints, per size class of the
plan, the mean duration of each phase over the class's blocks (microseconds) and, for cluster classes, rank 0 and the
other ranks apart.  A diagnostic: nothing here is on the solve path, and the numbers of the instrumented solve are not
bench values (profiles/r2_phases.md holds one such report).
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def report(cfg: int, scale: float = 1.0, dtype: str = "f64", steps: int = 20, out=sys.stdout, **plan_kw):
    import torch

    import morphgen as mg
    import paper_1810_12742_b200 as hb

    npd = np.float64 if dtype == "f64" else np.float32
    m = mg.make_config(cfg, scale)
    d, u, b = mg.system(m)
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == "f64" else hb.F32, **plan_kw)
    dd, du, db = (torch.from_numpy(a.astype(npd)).cuda() for a in (d, u, b))
    x = torch.empty_like(db)
    for _ in range(3):
        plan.solve(dd, du, db, x)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        plan.solve(dd, du, db, x)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    info = plan.info
    try:
        peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        peak = 6650.0
    print(f"== cfg{cfg} {dtype} {plan_kw}: {ms * 1e3:.1f} us/step, frac {info.bytes_min / ms / 1e6 / peak:.3f}, "
          f"blocks {info.n_blocks}", file=out)
    plan.enable_phase_clocks(True)
    plan.solve(dd, du, db, x)
    torch.cuda.synchronize()
    pc = plan.phase_clocks().astype(np.int64)
    first, count = plan.table("class_first"), plan.table("class_count")
    cl, sm = plan.table("class_cluster"), plan.table("class_smem_bytes")
    th, ph = plan.table("class_threads"), plan.table("class_phase")
    t0 = pc[:, 0].min()
    for q in range(len(first)):
        r = pc[first[q]:first[q] + count[q]]
        if not len(r):
            continue
        dur = np.diff(r[:, :7], axis=1) / 1e3
        unk = r[:, 7] & 0xffffffff
        print(f" class {q}: cl={cl[q]} smem={sm[q]} thr={th[q]} phase={ph[q]} blocks={count[q]} "
              f"unk/blk={unk.mean():.0f} start {(r[:, 0].min() - t0) / 1e3:.1f} end {(r[:, 6].max() - t0) / 1e3:.1f} us | "
              f"load {dur[:, 0].mean():.2f} P1 {dur[:, 1].mean():.2f} bwd {dur[:, 2].mean():.2f} "
              f"xch+fwd {dur[:, 3].mean():.2f} P3 {dur[:, 4].mean():.2f} store {dur[:, 5].mean():.2f} "
              f"total {(r[:, 6] - r[:, 0]).mean() / 1e3:.2f}", file=out)
        if cl[q] > 1:
            rr = r.reshape(-1, cl[q], 8)
            d0 = np.diff(rr[:, 0, :7], axis=1).mean(axis=0) / 1e3
            d1 = np.diff(rr[:, 1:, :7], axis=2).mean(axis=(0, 1)) / 1e3
            print(f"    rank0: load {d0[0]:.2f} P1 {d0[1]:.2f} bwd(incl wait) {d0[2]:.2f} fwd {d0[3]:.2f} "
                  f"P3 {d0[4]:.2f} store {d0[5]:.2f} | ranks>0: load {d1[0]:.2f} P1 {d1[1]:.2f} bwd {d1[2]:.2f} "
                  f"xch(wait) {d1[3]:.2f} P3 {d1[4]:.2f} store {d1[5]:.2f}", file=out)
    plan.close()


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.splitlines()[0])
    ap.add_argument("--config", type=int, nargs="+", default=[3])
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--dtype", choices=("f64", "f32"), default="f64")
    ap.add_argument("--steps", type=int, default=20)
    a = ap.parse_args(argv)
    for c in a.config:
        report(c, a.scale, a.dtype, a.steps)


if __name__ == "__main__":
    main()
