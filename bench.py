#!/usr/bin/env python
"""bench.py -- the batched Hines solve on B200: unknowns solved per second and achieved HBM GB/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--dtype f64|f32] [--impl ours|reference]

A "step" is one pass of the whole hot path (hines_solve: load, backward elimination, hand-off, root
solve, forward substitution, store) over one batch of synthetic input
(BASELINE.json config C, seeded, morphgen/).  Prints ONE JSON line (rank 0).

  value      whole-job unknowns/s with inputs resident in HBM (CUDA events on the launching stream,
             barrier + synchronize on both sides, max over ranks)
  e2e        the same through hines_solve_host: pinned HOST buffers, H2D of d,u,b and D2H of x inside
             the timed region every step
  roofline   HBM: algorithmic bytes (bytes_min = N*4w + 4*branches) / device time of the kernels of one
             step, against MEASURED_PEAKS.json hbm_gbs
  cpu_baseline  the oracle as it stands, timed on this box's host cores (rank 0, N=1 only)

N > 1 (torchrun): cells are independent, so each rank solves its own batch of the same
size with no collective on the data path: weak scaling.
--impl reference: times the CPU oracle (oracle/) on the same config and metric.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import morphgen as mg  # noqa: E402

METRIC = "hines_unknowns_solved_per_sec"
UNIT = "unknowns/s"
L2_BYTES = 126 * 1024 * 1024
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback


def peak_hbm():
    try:
        p = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload(cfg: int, scale: float, rank: int):
    seed = mg.rng.BASE_SEED + 7919 * rank           # every rank its own cells
    m = mg.make_config(cfg, scale, seed)
    d, u, _ = mg.coefficients(m, seed)
    b = mg.rhs(m, seed, 0)
    return m, d, u, b, seed


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the GPU is under load."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, windows):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if any(a <= t <= b for a, b in windows)] or [r for _, r in self.rows]
        sm, mx, pw, reasons = [], [], [], set()
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v == "Active":
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def cpu_oracle_time(m, d, u, b, threads: int, reps: int):
    """Best-of-`reps` seconds for the oracle over the whole batch with `threads` threads
    (plain parallel-for over cells: the ctypes call releases the GIL)."""
    import oracle
    d = np.ascontiguousarray(d, np.float64); u = np.ascontiguousarray(u, np.float64); b = np.ascontiguousarray(b, np.float64)
    par = np.ascontiguousarray(m.parent, np.int32); offs = np.ascontiguousarray(m.cell_offsets, np.int64)
    x = np.empty_like(d); dw = np.empty_like(d)
    # contiguous cell ranges of roughly equal unknowns
    cuts = np.searchsorted(offs, np.linspace(0, m.n, threads + 1)[1:-1]).tolist()
    bounds = [0] + cuts + [m.ncells]
    jobs = [(bounds[i], bounds[i + 1]) for i in range(threads) if bounds[i + 1] > bounds[i]]
    best = float("inf")
    with ThreadPoolExecutor(max_workers=max(1, len(jobs))) as ex:
        for _ in range(reps + 1):                    # first pass = warm-up
            t0 = time.perf_counter()
            list(ex.map(lambda j: oracle.hines_solve_range(j[0], j[1], par, offs, d, u, b, x, dw), jobs))
            dt = time.perf_counter() - t0
            best = min(best, dt) if _ else float("inf")
    return best, len(jobs), x


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    m, d, u, b, _ = workload(args.config, args.scale, 0)
    cores = os.cpu_count() or 1
    times = []
    for i in range(args.warmup + args.steps):
        t, used, _ = cpu_oracle_time(m, d, u, b, cores, 1)
        if i >= args.warmup:
            times.append(t)
    tot = sum(times)
    value = m.n * len(times) / tot
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": mg.CONFIG_NAMES[args.config], "scale": args.scale, "unknowns": m.n, "cells": m.ncells},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle",
                         "sample": "whole workload per step, parallel-for over cells (oracle/hines_oracle.c as it stands)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
def reduce_over_ranks(ms: float, e2e_s_per_step: float, units: float, dist=None, device="cpu"):
    """Whole-job numbers from per-rank ones: time = MAX over ranks, units = SUM over ranks.
    Cells are independent: this is the only communication of a multi-GPU run, and it
    is outside the timed region.  Works on any backend (nccl on GPUs, gloo in the CPU test)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms, e2e_s_per_step, units
    import torch
    t = torch.tensor([ms, e2e_s_per_step], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(n[0])


def measure(cfg, dtype, steps, warmup, rank, args, want_e2e, want_parity, barrier):
    """One config on this rank's GPU: device-resident timing, per-path device time, optional e2e."""
    import torch
    import paper_1810_12742_b200 as hb
    np_dtype = np.float64 if dtype == "f64" else np.float32
    w = np.dtype(np_dtype).itemsize
    m, d, u, b, seed = workload(cfg, args.scale, rank)
    t0 = time.perf_counter()
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == "f64" else hb.F32,
                   threads_per_block=args.threads, policy_flags=args.policy, group_smem_bytes=args.group_smem,
                   smem_bytes_per_block=args.smem, max_segment=args.max_segment, chunk_smem_bytes=args.chunk_smem,
                   cluster_max=args.cluster_max)
    plan.upload()
    plan_s = time.perf_counter() - t0
    info = plan.info
    bytes_min = info.bytes_min
    # device-resident inputs.  Working sets smaller than L2 rotate through > 2x L2 of distinct buffer
    # sets so that no step finds its inputs in L2 ("cold"); larger ones exceed L2 by themselves.
    nsets = 1 if bytes_min > L2_BYTES else min(64, int(np.ceil(2 * L2_BYTES / max(bytes_min, 1))) + 1)
    dd = torch.from_numpy(d.astype(np_dtype)).cuda()
    du = torch.from_numpy(u.astype(np_dtype)).cuda()
    sets = []
    for s in range(nsets):
        bs = b if s == 0 else mg.rhs(m, seed, s)              # fresh b per set (config 4: per time step)
        sets.append((dd if s == 0 else dd.clone(), du if s == 0 else du.clone(),
                     torch.from_numpy(bs.astype(np_dtype)).cuda(), torch.empty(m.n, dtype=dd.dtype, device="cuda")))
    stream = torch.cuda.current_stream().cuda_stream

    def step(i):
        a = sets[i % nsets]
        plan.solve(a[0], a[1], a[2], a[3], stream)

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    # ---- timed region: exactly `steps` steps, CUDA events on the launching stream -----------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    w0 = time.time()
    e0.record()
    for i in range(steps):
        step(i)
    e1.record()
    torch.cuda.synchronize(); barrier()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    windows = [(w0, w1)]
    # ---- parity of what was just timed (full batch, against the oracle) -----------------------
    parity = None
    if want_parity:
        import oracle
        dr, ur, br = (a.cpu().numpy().astype(np.float64) for a in sets[0][:3])
        xr = oracle.hines_solve(m.parent, m.cell_offsets, dr, ur, br)
        parity = float(oracle.rel_err(m.cell_offsets, sets[0][3].cpu().numpy().astype(np.float64), xr).max())
    # ---- per-path device time (roofline): the library's event hook, events on the same stream ----
    plan.enable_timing(True)
    res_ms, str_ms = [], []
    w2 = time.time()
    for i in range(min(steps, 50)):
        step(i)
        r_, s_ = plan.timing()
        res_ms.append(r_); str_ms.append(s_)
    w3 = time.time()
    plan.enable_timing(False)
    windows.append((w2, w3))
    res_ms, str_ms = float(np.mean(res_ms)), float(np.mean(str_ms))
    # ---- end to end: pinned host buffers through hines_solve_host -----------------------------
    e2e = None
    if want_e2e:
        hd, hu, hb_, hx = (torch.from_numpy(np.ascontiguousarray(a, np_dtype)).pin_memory() for a in (d, u, b, np.empty_like(b)))
        k_e2e = max(3, min(steps, int(np.ceil(3e9 / max(4 * m.n * w, 1)))))    # ~3 GB of traffic
        for _ in range(2):
            plan.solve_host(hd, hu, hb_, hx, stream)
        barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            plan.solve_host(hd, hu, hb_, hx, stream)
        e2e_s = (time.perf_counter() - t0) / k_e2e
        barrier()
        e2e = {"s_per_step": e2e_s, "steps": k_e2e, "h2d": 3 * m.n * w, "d2h": m.n * w}
    launches = plan.launches_per_solve
    out = {"m": m, "d": d, "u": u, "b": b, "info": info, "ms": ms, "res_ms": res_ms, "str_ms": str_ms,
           "parity": parity, "e2e": e2e, "plan_s": plan_s, "nsets": nsets, "launches": launches,
           "windows": windows, "bytes_min": bytes_min, "bytes_literal": info.bytes_literal,
           "classes": [int(v) for v in plan.table("class_cluster")]}
    plan.close()
    del sets, dd, du
    torch.cuda.empty_cache()
    return out


def load_traffic(key):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per step, from the committed
    ncu --set full capture (profiles/traffic.csv, see profiles/traffic.md), or None."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "traffic.csv")).read().splitlines()[1:]:
            k, v = line.split(",")
            if k == key:
                return int(v)
    except Exception:
        pass
    return None


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs[] index (default 1)")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of the other configs")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--policy", type=int, default=0)
    ap.add_argument("--group-smem", type=int, default=0)
    ap.add_argument("--smem", type=int, default=0)
    ap.add_argument("--max-segment", type=int, default=0)
    ap.add_argument("--chunk-smem", type=int, default=0)
    ap.add_argument("--cluster-max", type=int, default=0)
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()

    sampler = ClockSampler(local) if rank == 0 else None
    r = measure(args.config, args.dtype, args.steps, args.warmup, rank, args,
                want_e2e=not args.no_e2e, want_parity=(rank == 0 and not args.no_cpu), barrier=barrier)
    clocks = sampler.stop(r["windows"]) if sampler else None
    m, info = r["m"], r["info"]
    ms, e2e_s, tot_units = reduce_over_ranks(r["ms"], r["e2e"]["s_per_step"] if r["e2e"] else 0.0, float(m.n),
                                             dist if world > 1 else None, "cuda")

    # the other configs, short runs (parity-test cases, not bench lines): context for the headline
    others = {}
    if not args.no_others and world == 1 and args.scale == 1.0:
        for cfg, dt in ((0, "f64"), (1, "f64"), (2, "f64"), (2, "f32"), (3, "f64"), (4, "f64")):
            if cfg == args.config and dt == args.dtype:
                continue
            try:
                o = measure(cfg, dt, min(args.steps, 20), 3, rank, args, False, False, barrier)
                others[f"cfg{cfg}_{dt}"] = {
                    "unknowns": o["m"].n, "ms_per_step": o["ms"] / min(args.steps, 20),
                    "value": o["m"].n * min(args.steps, 20) / (o["ms"] * 1e-3),
                    "hbm_frac": o["bytes_min"] / (o["ms"] / min(args.steps, 20) * 1e-3) / 1e9 / peak_hbm()[0],
                    "resident_ms": o["res_ms"], "stream_ms": o["str_ms"], "launches_per_step": o["launches"],
                    "cluster_sizes": o["classes"], "stream_cells": o["info"].n_stream_cells}
                del o
            except Exception as ex:                       # a context line must never kill the headline
                others[f"cfg{cfg}_{dt}"] = {"error": str(ex)[:200]}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    w = 8 if args.dtype == "f64" else 4
    ms_step = ms / args.steps
    value = tot_units * args.steps / (ms * 1e-3)
    peak, peak_src = peak_hbm()
    res_ms, str_ms = r["res_ms"], r["str_ms"]
    # The launches of one step are one kernel family (resident: one launch per size class, overlapping on side
    # streams; or the streaming pair, one launch per level) and fill the step: their average duration over the
    # timed region is the region divided by its steps.  res_ms / str_ms (one isolated step at a time, through
    # the library's event hook, so each includes a cold start) say which path dominates.
    achieved = r["bytes_min"] / (ms_step * 1e-3) / 1e9
    dominant = "hines_resident_kernel" if res_ms >= str_ms else "hines_stream_backward/forward"

    cpu = None
    if not args.no_cpu and world == 1:
        cores = os.cpu_count() or 1
        # bounded sample: whole cells from the start of the batch, at most ~40 M unknowns
        ncs = int(np.searchsorted(m.cell_offsets, min(m.n, 40_000_000), side="left"))
        ncs = max(1, min(ncs, m.ncells))
        ms_ = mg.Morphology(m.parent[:m.cell_offsets[ncs]], m.cell_offsets[:ncs + 1])
        ns = ms_.n
        t1, _, _ = cpu_oracle_time(ms_, r["d"][:ns], r["u"][:ns], r["b"][:ns], 1, 2)
        tn, used, _ = cpu_oracle_time(ms_, r["d"][:ns], r["u"][:ns], r["b"][:ns], cores, 5)
        cpu = {"value": ns / tn, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"first {ncs} cells ({ns} unknowns) of the workload, best of 5 after warm-up, parallel-for over cells",
               "single_thread_value": ns / t1, "cpu_count": cores}

    e2e = r["e2e"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": mg.CONFIG_NAMES[args.config], "scale": args.scale, "unknowns_per_gpu": m.n,
                   "cells_per_gpu": m.ncells, "branches_per_gpu": info.nbranches, "max_levels": info.max_levels,
                   "parallelism": f"independent cells, {world} replica(s), no collective",
                   "l2": "inputs_exceed_l2" if r["nsets"] == 1 else f"rotating {r['nsets']} distinct buffer sets (> 2x L2)",
                   "resident_items": info.n_resident_items, "resident_blocks": info.n_blocks,
                   "resident_unknowns": info.n_resident_unknowns, "cluster_cells": info.n_cluster_cells,
                   "cluster_unknowns": info.n_cluster_unknowns, "cluster_sizes_per_class": r["classes"],
                   "stream_cells": info.n_stream_cells, "stream_unknowns": info.n_stream_unknowns,
                   "size_classes": info.n_classes,
                   "lane_efficiency": info.useful_lane_steps / max(1, info.padded_lane_steps),
                   "plan_create_s": r["plan_s"]},
        "achieved_hbm_gbs": r["bytes_min"] * world / (ms_step * 1e-3) / 1e9,
        "hbm_frac_of_peak_per_gpu": r["bytes_min"] / (ms_step * 1e-3) / 1e9 / peak,
        "bytes_min_per_step": r["bytes_min"], "bytes_literal_per_step": r["bytes_literal"],
        "gpu_launches": r["launches"] * args.steps,
        "clocks": clocks,
        "e2e": None if e2e is None else {"value": tot_units / e2e_s, "unit": UNIT, "steps": e2e["steps"],
                                         "h2d_bytes_per_step": e2e["h2d"] * world, "d2h_bytes_per_step": e2e["d2h"] * world},
        "roofline": {"bound": "hbm", "kernel": dominant, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": load_traffic(f"cfg{args.config}_{args.dtype}"),
                     "peak_source": peak_src, "resident_ms": res_ms, "stream_ms": str_ms,
                     "note": "achieved = bytes_min (N*4w + 4*branches, all launches of one step) / average device time "
                             "of one step's launches over the timed region (CUDA events on the launching stream); "
                             "resident_ms / stream_ms = one isolated step per path (library event hook, cold start)"},
        "cpu_baseline": cpu,
        "parity_max_rel_err": r["parity"],
        "other_configs": others,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
