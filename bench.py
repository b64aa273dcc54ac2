#!/usr/bin/env python
"""bench.py -- the batched Hines solve on B200: unknowns solved per second and achieved HBM GB/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--dtype f64|f32] [--impl ours|reference]

A "step" is one pass of the whole hot path (hines_solve: load, backward elimination, hand-off, root
solve, forward substitution, store) over one batch of synthetic input
(BASELINE.json config C, seeded, morphgen/).  Default config: 3, the largest single-GPU configuration
(BASELINE.json's metric names none).  Prints ONE JSON line (rank 0).

  value      whole-job unknowns/s with inputs resident in HBM: exactly K steps between two CUDA events on the
             launching stream, barrier + synchronize on both sides, max over ranks
  timing     the same in >= 20 intervals of >= 50 ms each: median and best ms per step
  e2e        the same through hines_host_pipeline_solve: pinned HOST buffers, H2D of d,u,b and D2H of x inside
             the timed region every step (slices of whole cells, copies and solves overlapped; the figure of the
             one-call hines_solve_host beside it)
  roofline   HBM: algorithmic bytes (bytes_min = N*4w + 4*branches) / device time of the kernels of one
             step, against MEASURED_PEAKS.json hbm_gbs
  cpu_baseline  the oracle as it stands, timed on this box's host cores (rank 0, N=1 only)
  other_configs the remaining configs, each with its own roofline / parity / clocks block

N > 1 (torchrun): cells are independent, so each rank solves its own batch of the same
size with no collective on the data path: weak scaling.
--impl reference: times the CPU oracle (oracle/) on the same config and metric.
"""
from __future__ import annotations

import argparse
import hashlib
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
INTERVAL_MS = 50.0            # every timed interval at least this long
N_INTERVALS = 20


def peak_hbm():
    try:
        p = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload(cfg: int, scale: float, rank: int, world: int = 1, scaling: str = "weak"):
    """This rank's cells.  weak: every rank generates its own batch of the config's size (seed offset by rank).
    strong: ONE batch of the config's size, its cells dealt to the ranks by hines_partition_cells (longest processing
    time first on the cells' unknowns); the rank keeps its cells in input order."""
    if scaling == "weak" or world == 1:
        seed = mg.rng.BASE_SEED + 7919 * rank       # every rank its own cells
        m = mg.make_config(cfg, scale, seed)
        d, u, _ = mg.coefficients(m, seed)
        b = mg.rhs(m, seed, 0)
        return m, d, u, b, seed
    seed = mg.rng.BASE_SEED
    m = mg.make_config(cfg, scale, seed)
    d, u, _ = mg.coefficients(m, seed)
    b = mg.rhs(m, seed, 0)
    ms, idx = my_share(m, rank, world)
    return ms, d[idx], u[idx], b[idx], seed


def my_share(m, rank: int, world: int):
    """(sub-morphology, compartment indices) of the cells hines_partition_cells gives to `rank` of `world`."""
    import paper_1810_12742_b200 as hb
    part, _ = hb.partition_cells(m.cell_offsets, world)
    mine = np.nonzero(part == rank)[0]
    lo, hi = m.cell_offsets[mine], m.cell_offsets[mine + 1]
    idx = np.concatenate([np.arange(a, b_) for a, b_ in zip(lo, hi)]) if len(mine) else np.zeros(0, np.int64)
    offs = np.concatenate([[0], np.cumsum(hi - lo)]).astype(np.int64)
    ms = mg.Morphology(m.parent[idx], offs, name=m.name)
    ms.meta["cells"] = mine
    return ms, idx


def config_block(cfg: int, scale: float, m):
    """The keys both arms print under "config" (identical in the two arms)."""
    return {"workload": mg.CONFIG_NAMES[cfg], "scale": scale, "unknowns": int(m.n), "cells": int(m.ncells)}


def kernel_hash() -> str:
    """Identifies the kernel + planner sources a measured traffic figure belongs to."""
    h = hashlib.sha256()
    for f in ("paper_1810_12742_b200/csrc/solve.cu", "paper_1810_12742_b200/csrc/plan.cpp",
              "paper_1810_12742_b200/csrc/plan_internal.h"):
        h.update(open(os.path.join(ROOT, f), "rb").read())
    return h.hexdigest()[:16]


def load_traffic(key):
    """dram__bytes_read.sum + dram__bytes_write.sum of all kernels of one step, from a committed ncu capture
    (profiles/traffic.csv: key,bytes,source_hash,command; see profiles/traffic.md) -- or None when that capture
    was made with other kernel sources than the ones in the tree (it would be stale)."""
    try:
        cur = kernel_hash()
        for line in open(os.path.join(ROOT, "profiles", "traffic.csv")).read().splitlines()[1:]:
            f = line.split(",", 3)
            if f[0] == key and f[2] == cur:
                return int(f[1])
    except Exception:
        pass
    return None


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
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20", "-i", str(index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def summary(self, windows):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        rows = [r for (t, r) in list(self.rows) if any(a <= t <= b for a, b in windows)]
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

    def stop(self):
        if self.proc is not None:
            time.sleep(0.05)
            self.proc.terminate()


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


def head_sample(m, d, u, b, max_unknowns):
    """Whole cells from the start of the batch, at most max_unknowns (at least one cell)."""
    ncs = int(np.searchsorted(m.cell_offsets, min(m.n, max_unknowns), side="right")) - 1
    ncs = max(1, min(ncs, m.ncells))
    ns = int(m.cell_offsets[ncs])
    return mg.Morphology(m.parent[:ns], m.cell_offsets[:ncs + 1]), d[:ns], u[:ns], b[:ns], ncs


def sampled_parity(m, d, u, b, x_gpu, np_dtype, max_unknowns=12_000_000):
    """Max per-cell relative max-norm error of the GPU solution against the oracle (reading S15), on every cell when
    the batch is small, else on every k-th cell (about max_unknowns unknowns): the oracle solves exactly those cells."""
    import oracle
    k = max(1, int(np.ceil(m.n / max_unknowns)))
    sel = np.arange(0, m.ncells, k)
    lo, hi = m.cell_offsets[sel], m.cell_offsets[sel + 1]
    idx = np.concatenate([np.arange(a, b_) for a, b_ in zip(lo, hi)]) if k > 1 else slice(None)
    offs = np.concatenate([[0], np.cumsum(hi - lo)]).astype(np.int64)
    rd = lambda a: np.ascontiguousarray(a[idx], np_dtype).astype(np.float64)       # the oracle sees the rounded inputs
    xr = oracle.hines_solve(m.parent[idx], offs, rd(d), rd(u), rd(b))
    xg = np.ascontiguousarray(x_gpu[idx], np.float64)
    finite = bool(np.isfinite(x_gpu).all())
    err = float(oracle.rel_err(offs, xg, xr).max())
    return {"max_rel_err": err if finite else float("nan"), "finite": finite, "cells_checked": int(len(sel)),
            "unknowns_checked": int(offs[-1]), "every_kth_cell": k}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    m, d, u, b, _ = workload(args.config, args.scale, 0)
    cores = os.cpu_count() or 1
    ms_, ds, us, bs, ncs = head_sample(m, d, u, b, 40_000_000)     # bounded sample of the workload per step
    times, used = [], 1
    for i in range(args.warmup + args.steps):
        t, used, _ = cpu_oracle_time(ms_, ds, us, bs, cores, 1)
        if i >= args.warmup:
            times.append(t)
    tot = sum(times)
    value = ms_.n * len(times) / tot
    sample = (f"each step = the first {ncs} cells ({ms_.n} unknowns) of the workload, parallel-for over cells "
              f"(oracle/hines_oracle.c as it stands)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_block(args.config, args.scale, m),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
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


def measure(cfg, dtype, steps, warmup, rank, args, want_e2e, want_parity, barrier, intervals=N_INTERVALS):
    """One config on this rank's GPU: exactly `steps` timed steps, then `intervals` intervals of >= 50 ms, the
    per-path device time, parity of what was timed, optional e2e."""
    import torch
    import paper_1810_12742_b200 as hb
    np_dtype = np.float64 if dtype == "f64" else np.float32
    w = np.dtype(np_dtype).itemsize
    m, d, u, b, seed = workload(cfg, args.scale, rank, args.world, args.scaling)
    t0 = time.perf_counter()
    plan_kw = dict(threads_per_block=args.threads, policy_flags=args.policy, group_smem_bytes=args.group_smem,
                   smem_bytes_per_block=args.smem, max_segment=args.max_segment, chunk_smem_bytes=args.chunk_smem,
                   cluster_max=args.cluster_max, split_smem_bytes=args.split_smem)
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == "f64" else hb.F32, **plan_kw)
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

    # Launch-bound configs (a step of a few tens of microseconds: config 4's time loop, config 0) are replayed as a
    # CUDA graph of one pass over the buffer sets, as SURVEY.md section 8(d) asks ("the 1,000 steps as one graph launch").
    use_graph = nsets > 1 and not args.no_graph
    graph = None
    if use_graph:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            for i in range(nsets):
                a = sets[i]
                plan.solve(a[0], a[1], a[2], a[3], side.cuda_stream)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            for i in range(nsets):
                a = sets[i]
                plan.solve(a[0], a[1], a[2], a[3], side.cuda_stream)

    def run_steps(k):
        """k steps on the current stream (graph: whole passes over the buffer sets, k rounded up to one)."""
        if graph is None:
            for i in range(k):
                step(i)
            return k
        n = -(-k // nsets)
        for _ in range(n):
            graph.replay()
        return n * nsets

    run_steps(max(warmup, 3))
    torch.cuda.synchronize()
    # ---- timed region: exactly `steps` steps, CUDA events on the launching stream -----------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    w0 = time.time()
    e0.record()
    done = run_steps(steps)
    e1.record()
    torch.cuda.synchronize(); barrier()
    ms = e0.elapsed_time(e1) * steps / done                   # (graph replays are whole passes: scaled to `steps`)
    # ---- >= 20 intervals of >= 50 ms each: median and best ------------------------------------
    per_step = ms / steps
    inner = max(1, int(np.ceil(INTERVAL_MS / max(per_step, 1e-6))))
    iv = []
    for _ in range(0 if args.no_intervals else intervals):
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        n_ = run_steps(inner)
        a1.record()
        a1.synchronize()
        iv.append(a0.elapsed_time(a1) / n_)
    w1 = time.time()
    windows = [(w0, w1)]
    timing = {"intervals": intervals, "steps_per_interval": inner, "interval_ms": float(np.median(iv)) * inner,
              "median_ms_per_step": float(np.median(iv)), "best_ms_per_step": float(np.min(iv)),
              "worst_ms_per_step": float(np.max(iv))} if iv else None
    # ---- parity of what was just timed (against the oracle, on the cells the oracle is given) ----
    parity = None
    if want_parity:
        step(0); torch.cuda.synchronize()
        parity = sampled_parity(m, d, u, b, sets[0][3].cpu().numpy(), np_dtype)
    # ---- per-path device time: the library's event hook ----------------------------------------
    plan.enable_timing(True)
    res_ms, str_ms = [], []
    for i in range(1 if args.no_intervals else 10):
        step(i)
        r_, s_ = plan.timing()
        res_ms.append(r_); str_ms.append(s_)
    plan.enable_timing(False)
    res_ms, str_ms = float(np.mean(res_ms)), float(np.mean(str_ms))
    # ---- end to end: pinned host buffers through hines_solve_host -----------------------------
    e2e = None
    if want_e2e:
        hd, hu, hb_, hx = (torch.from_numpy(np.ascontiguousarray(a, np_dtype)).pin_memory() for a in (d, u, b, np.empty_like(b)))
        k_e2e = max(3, min(steps, int(np.ceil(3e9 / max(4 * m.n * w, 1)))))    # ~3 GB of traffic

        def timed(call):
            for _ in range(2):
                call()
            barrier()
            t0 = time.perf_counter()
            for _ in range(k_e2e):
                call()
            dt = (time.perf_counter() - t0) / k_e2e
            barrier()
            return dt
        # one call, the link busy in one direction at a time ...
        single_s = timed(lambda: plan.solve_host(hd, hu, hb_, hx, stream))
        x_single = hx.numpy().copy()
        # ... and the pipelined entry: slices of whole cells, copy-in / solve / copy-out overlapped (the e2e figure)
        pipe = hb.HostPipeline(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == "f64" else hb.F32, **plan_kw)
        hx.fill_(float("nan"))
        e2e_s = timed(lambda: pipe.solve(hd, hu, hb_, hx))
        x_pipe = hx.numpy()
        scale_ = np.abs(x_single).max()
        e2e = {"s_per_step": e2e_s, "steps": k_e2e, "h2d": 3 * m.n * w, "d2h": m.n * w,
               "entry": f"hines_host_pipeline_solve ({len(pipe.slices) - 1} slices)", "single_call_s_per_step": single_s,
               "max_abs_diff_vs_single_call_over_max_abs_x": float(np.abs(x_pipe - x_single).max() / scale_)}
        assert np.isfinite(x_pipe).all() and e2e["max_abs_diff_vs_single_call_over_max_abs_x"] < (1e-10 if w == 8 else 1e-4)
        pipe.close()
        del hd, hu, hb_, hx
    out = {"m": m, "d": d, "u": u, "b": b, "info": info, "ms": ms, "res_ms": res_ms, "str_ms": str_ms,
           "parity": parity, "e2e": e2e, "plan_s": plan_s, "nsets": nsets, "launches": plan.launches_per_solve,
           "windows": windows, "bytes_min": bytes_min, "bytes_literal": info.bytes_literal, "timing": timing,
           "graph": graph is not None,
           "classes": [int(v) for v in plan.table("class_cluster")], "phases": [int(v) for v in plan.table("class_phase")]}
    del graph
    plan.close()
    del sets, dd, du
    torch.cuda.empty_cache()
    return out


def measure_factored(cfg, dtype, steps, rank, args, want_parity):
    """f3: hines_factor once, then `steps` hines_solve_rhs calls with a fresh b per step, device-resident.
    Roofline numerator of this entry: the factors (3w) + b (w) read, x (w) written = 5*N*w + 4*branches."""
    import torch
    import paper_1810_12742_b200 as hb
    np_dtype = np.float64 if dtype == "f64" else np.float32
    w = np.dtype(np_dtype).itemsize
    m, d, u, b, seed = workload(cfg, args.scale, rank, args.world, args.scaling)
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == "f64" else hb.F32, policy_flags=args.policy | hb.POLICY_FACTORED)
    info = plan.info
    if info.n_stream_cells:
        plan.close()
        return {"error": "cells on the streaming path"}
    dd, du = (torch.from_numpy(a.astype(np_dtype)).cuda() for a in (d, u))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    plan.factor(dd, du); torch.cuda.synchronize()
    e0.record(); plan.factor(dd, du); e1.record(); torch.cuda.synchronize()
    factor_ms = e0.elapsed_time(e1)
    del dd, du
    bytes_rhs = 5 * m.n * w + 4 * info.nbranches
    nsets = 1 if bytes_rhs > L2_BYTES else min(64, int(np.ceil(2 * L2_BYTES / max(2 * m.n * w, 1))) + 1)
    sets = [(torch.from_numpy((b if s == 0 else mg.rhs(m, seed, s)).astype(np_dtype)).cuda(),
             torch.empty(m.n, dtype=torch.float64 if dtype == "f64" else torch.float32, device="cuda")) for s in range(nsets)]
    stream = torch.cuda.current_stream().cuda_stream
    graph = None
    if nsets > 1 and not args.no_graph:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            for bb, xx in sets:
                plan.solve_rhs(bb, xx, side.cuda_stream)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            for bb, xx in sets:
                plan.solve_rhs(bb, xx, side.cuda_stream)

    def run_steps(k):
        if graph is None:
            for i in range(k):
                plan.solve_rhs(sets[i % nsets][0], sets[i % nsets][1], stream)
            return k
        n = -(-k // nsets)
        for _ in range(n):
            graph.replay()
        return n * nsets

    run_steps(5); torch.cuda.synchronize()
    e0.record(); done = run_steps(steps); e1.record(); torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / done
    inner = max(1, int(np.ceil(INTERVAL_MS / max(ms_step, 1e-6))))
    iv = []
    for _ in range(N_INTERVALS):
        e0.record(); n_ = run_steps(inner); e1.record(); e1.synchronize()
        iv.append(e0.elapsed_time(e1) / n_)
    parity = None
    if want_parity:
        plan.solve_rhs(sets[0][0], sets[0][1], stream); torch.cuda.synchronize()
        parity = sampled_parity(m, d, u, b, sets[0][1].cpu().numpy(), np_dtype)["max_rel_err"]
    peak, _ = peak_hbm()
    out = {"entry": "hines_factor once + hines_solve_rhs per step (fresh b per step)", "ms_per_step": ms_step,
           "median_ms_per_step": float(np.median(iv)), "best_ms_per_step": float(np.min(iv)),
           "value": m.n / (ms_step * 1e-3), "unit": UNIT, "factor_ms": factor_ms, "cuda_graph": graph is not None,
           "bytes_per_step": bytes_rhs, "achieved_gbs": bytes_rhs / (ms_step * 1e-3) / 1e9,
           "frac_of_peak": bytes_rhs / (ms_step * 1e-3) / 1e9 / peak, "launches_per_step": plan.launches_per_solve,
           "parity_max_rel_err": parity}
    del graph, sets
    plan.close()
    torch.cuda.empty_cache()
    return out


def plan_block(r, world):
    info = r["info"]
    return {"branches": info.nbranches, "max_levels": info.max_levels,
            "parallelism": f"independent cells, {world} replica(s), no collective",
            "l2": "inputs_exceed_l2" if r["nsets"] == 1 else f"rotating {r['nsets']} distinct buffer sets of d,u,b,x (> 2x L2): cold",
            "cuda_graph": r["graph"], "resident_items": info.n_resident_items, "parts": info.n_parts,
            "blocks_per_step": info.n_blocks, "cluster_cells": info.n_cluster_cells,
            "cluster_unknowns": info.n_cluster_unknowns, "split_cells": info.n_split_cells,
            "split_unknowns": info.n_split_unknowns, "exports": info.n_exports,
            "cluster_size_per_class": r["classes"], "phase_per_class": r["phases"],
            "stream_cells": info.n_stream_cells, "stream_unknowns": info.n_stream_unknowns,
            "launches_per_step": r["launches"],
            "lane_efficiency": info.useful_lane_steps / max(1, info.padded_lane_steps), "plan_create_s": r["plan_s"]}


def roofline_block(r, key, steps):
    peak, peak_src = peak_hbm()
    ms_step = r["ms"] / steps
    achieved = r["bytes_min"] / (ms_step * 1e-3) / 1e9
    best = r["bytes_min"] / (r["timing"]["median_ms_per_step"] * 1e-3) / 1e9 if r["timing"] else None
    dominant = "hines_resident_kernel" if r["res_ms"] >= r["str_ms"] else "hines_stream_backward/forward"
    return {"bound": "hbm", "kernel": dominant, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "frac_median_of_intervals": None if best is None else best / peak,
            "traffic": load_traffic(key), "peak_source": peak_src, "resident_ms": r["res_ms"], "stream_ms": r["str_ms"],
            "note": "achieved = bytes_min (N*4w + 4*branches, all launches of one step) / average device time of one step over "
                    "the timed region (CUDA events on the launching stream); one kernel family fills the step; resident_ms / "
                    "stream_ms = one isolated step per path (library event hook); traffic = measured DRAM bytes of one step from "
                    "the committed ncu capture of these very sources (profiles/traffic.csv), else null"}


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs[] index (default 3: the largest single-GPU one)")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the runs of the other configs")
    ap.add_argument("--no-factored", action="store_true", help="skip the hines_factor / hines_solve_rhs entry (f3)")
    ap.add_argument("--no-intervals", action="store_true", help="only the K timed steps (for runs under ncu)")
    ap.add_argument("--no-graph", action="store_true", help="launch-bound configs step by step instead of as a CUDA graph")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--policy", type=int, default=0)
    ap.add_argument("--group-smem", type=int, default=0)
    ap.add_argument("--smem", type=int, default=0)
    ap.add_argument("--max-segment", type=int, default=0)
    ap.add_argument("--chunk-smem", type=int, default=0)
    ap.add_argument("--cluster-max", type=int, default=0)
    ap.add_argument("--split-smem", type=int, default=0)
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own batch of the config size; strong = one batch, cells dealt to the ranks")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    args.world = 1
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    args.world = world
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
    clocks = sampler.summary(r["windows"]) if sampler else None
    m = r["m"]
    ms, e2e_s, tot_units = reduce_over_ranks(r["ms"], r["e2e"]["s_per_step"] if r["e2e"] else 0.0, float(m.n),
                                             dist if world > 1 else None, "cuda")

    # the other configs (parity-test cases, not bench lines): each with its own roofline / parity / clocks block
    others = {}
    if not args.no_others and world == 1 and args.scale == 1.0:
        for cfg, dt in ((0, "f64"), (1, "f64"), (2, "f64"), (2, "f32"), (3, "f64"), (4, "f64")):
            if cfg == args.config and dt == args.dtype:
                continue
            try:
                k = max(20, min(args.steps, 100))
                o = measure(cfg, dt, k, 5, rank, args, False, not args.no_cpu, barrier)
                others[f"cfg{cfg}_{dt}"] = {
                    "config": config_block(cfg, args.scale, o["m"]), "dtype": dt, "steps": k,
                    "ms_per_step": o["ms"] / k, "value": o["m"].n * k / (o["ms"] * 1e-3), "unit": UNIT,
                    "timing": o["timing"], "roofline": roofline_block(o, f"cfg{cfg}_{dt}", k),
                    "parity": o["parity"], "clocks": sampler.summary(o["windows"]) if sampler else None,
                    "bytes_min_per_step": o["bytes_min"], "gpu_launches": o["launches"] * k, "plan": plan_block(o, world)}
                del o
                if cfg in (3, 4) and not args.no_factored:
                    others[f"cfg{cfg}_{dt}"]["factored"] = measure_factored(cfg, dt, k, rank, args, not args.no_cpu)
            except Exception as ex:                       # a context line must never kill the headline
                others[f"cfg{cfg}_{dt}"] = {"error": str(ex)[:300]}
    factored = None
    if not args.no_factored and world == 1:
        try:
            factored = measure_factored(args.config, args.dtype, args.steps, rank, args, not args.no_cpu)
        except Exception as ex:
            factored = {"error": str(ex)[:300]}
    if sampler:
        sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms / args.steps
    value = tot_units * args.steps / (ms * 1e-3)
    roof = roofline_block(r, f"cfg{args.config}_{args.dtype}", args.steps)

    cpu = None
    if not args.no_cpu and world == 1:
        cores = os.cpu_count() or 1
        ms_, ds, us, bs, ncs = head_sample(m, r["d"], r["u"], r["b"], 40_000_000)      # bounded sample
        t1, _, _ = cpu_oracle_time(ms_, ds, us, bs, 1, 1)
        tn, used, _ = cpu_oracle_time(ms_, ds, us, bs, cores, 5)
        cpu = {"value": ms_.n / tn, "unit": UNIT, "cores": used, "kind": "oracle",
               "sample": f"first {ncs} cells ({ms_.n} unknowns) of the workload, best of 5 after warm-up, parallel-for over cells",
               "single_thread_value": ms_.n / t1, "cpu_count": cores}

    e2e = r["e2e"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
        "dtype": args.dtype, "data": "synthetic",
        "config": config_block(args.config, args.scale, m),
        "plan": plan_block(r, world),
        "timing": r["timing"],
        "achieved_hbm_gbs": r["bytes_min"] * world / (ms_step * 1e-3) / 1e9,
        "hbm_frac_of_peak_per_gpu": roof["frac"],
        "bytes_min_per_step": r["bytes_min"], "bytes_literal_per_step": r["bytes_literal"],
        "gpu_launches": r["launches"] * args.steps,
        "clocks": clocks,
        "e2e": None if e2e is None else {"value": tot_units / e2e_s, "unit": UNIT, "steps": e2e["steps"],
                                         "h2d_bytes_per_step": e2e["h2d"] * world, "d2h_bytes_per_step": e2e["d2h"] * world,
                                         "entry": e2e["entry"],
                                         "single_call_value_rank0": float(m.n) / e2e["single_call_s_per_step"],
                                         "max_abs_diff_vs_single_call_over_max_abs_x": e2e["max_abs_diff_vs_single_call_over_max_abs_x"]},
        "roofline": roof,
        "cpu_baseline": cpu,
        "factored": factored,
        "parity": r["parity"],
        "parity_max_rel_err": None if r["parity"] is None else r["parity"]["max_rel_err"],
        "kernel_source_hash": kernel_hash(),
        "other_configs": others,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
