"""Host logic of the multi-GPU bench path, on CPU with the gloo backend and world size 2:
every rank solves its own cells (cells are independent, no collective on the data
path); the only communication is the reduction of the timings (MAX) and of the units (SUM)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e, units = bench.reduce_over_ranks(10.0 + 5 * rank, 0.5 - 0.1 * rank, 1000.0 * (rank + 1), dist, "cpu")
    m, d, u, b, seed = bench.workload(0, 1.0, rank)
    out.put((rank, ms, e2e, units, seed, float(d[:16].sum())))
    dist.destroy_process_group()


def test_reduce_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, units, seed, dsum in res:
        assert ms == 15.0 and e2e == 0.5 and units == 3000.0          # MAX, MAX, SUM on every rank
    assert res[0][4] != res[1][4] and res[0][5] != res[1][5]          # every rank its own cells


def test_single_process_passthrough():
    import bench
    assert bench.reduce_over_ranks(1.5, 0.25, 42.0) == (1.5, 0.25, 42.0)


def test_reference_arm_prints_the_contract_line(capsys):
    import json
    import bench
    sys_argv = sys.argv
    sys.argv = ["bench.py", "--impl", "reference", "--config", "0", "--steps", "2", "--warmup", "3"]
    try:
        bench.main()
    finally:
        sys.argv = sys_argv
    line = json.loads(capsys.readouterr().out.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "unknowns/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"].startswith("cfg0") and line["higher_is_better"] is True
