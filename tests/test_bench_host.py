"""Host logic of the multi-GPU path, on CPU with the gloo backend and world size 2: ONE batch's cells are dealt to
the ranks by hines_partition_cells (longest processing time first on the cells' unknowns);
every rank plans ITS part of that same batch (hines_plan_create needs no device); the parts are disjoint, cover every
cell and are balanced; no collective touches the data path (cells are independent) -- the only
communication is the reduction of the timings (MAX) and of the units (SUM).  Config 4 (a single cell) cannot be
partitioned: replicas only."""
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
    import morphgen as mg
    import paper_1810_12742_b200 as hb
    ms, e2e, units = bench.reduce_over_ranks(10.0 + 5 * rank, 0.5 - 0.1 * rank, 1000.0 * (rank + 1), dist, "cpu")
    m, d, u, b, seed = bench.workload(0, 1.0, rank)                     # weak scaling: every rank its own batch
    # strong scaling: this rank's part of ONE heterogeneous batch (config 3, a slice), planned without a device
    ps, dps, ups, bps, _ = bench.workload(3, 0.01, rank, world, "strong")
    plan = hb.Plan(ps.parent, ps.cell_offsets)
    info = plan.info
    assert info.n == ps.n == len(dps) and info.n_resident_unknowns + info.n_stream_unknowns == ps.n
    out.put((rank, ms, e2e, units, seed, float(d[:16].sum()), ps.meta["cells"].tolist(), int(ps.n), float(dps.sum())))
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
    for rank, ms, e2e, units, seed, dsum, cells, n, dps in res:
        assert ms == 15.0 and e2e == 0.5 and units == 3000.0          # MAX, MAX, SUM on every rank
    assert res[0][4] != res[1][4] and res[0][5] != res[1][5]          # weak: every rank its own cells
    # strong: the two parts of the same batch are disjoint, cover every cell, and differ in cost by < 5 %
    import morphgen as mg
    import bench
    m = mg.make_config(3, 0.01)
    c0, c1 = set(res[0][6]), set(res[1][6])
    assert not (c0 & c1) and c0 | c1 == set(range(m.ncells))
    assert res[0][7] + res[1][7] == m.n and abs(res[0][7] - res[1][7]) < 0.05 * m.n / 2
    d, _, _ = mg.coefficients(m)
    assert abs(res[0][8] + res[1][8] - d.sum()) < 1e-6 * d.sum()       # every compartment's coefficients went to one rank


def test_partition_cells_lpt():
    """hines_partition_cells: longest processing time first, deterministic; every cell to exactly one device."""
    import paper_1810_12742_b200 as hb
    import morphgen as mg
    sizes = np.array([5, 100, 7, 100, 30, 1, 60, 2], np.int64)
    offs = np.concatenate([[0], np.cumsum(sizes)])
    part, cost = hb.partition_cells(offs, 3)
    # by hand: 100->0, 100->1, 60->2, 30->2, 7->2, 5->2, 2->0 (ties: lowest device among the lightest), 1->1
    assert part.tolist() == [2, 0, 2, 1, 2, 1, 2, 0] and cost.tolist() == [102, 101, 102]
    m = mg.make_config(3, 0.02)
    for n in (1, 2, 4, 8):
        part, cost = hb.partition_cells(m.cell_offsets, n)
        assert part.min() >= 0 and part.max() < n and cost.sum() == m.n
        assert np.array_equal(np.bincount(part, weights=np.diff(m.cell_offsets), minlength=n).astype(np.int64), cost)
        assert cost.max() - cost.min() <= np.diff(m.cell_offsets).max()       # the LPT bound
    with pytest.raises(hb.HinesError):
        hb.partition_cells(offs, 0)
    one = mg.make_config(4)                                             # config 4: one cell -> replicas only
    part, cost = hb.partition_cells(one.cell_offsets, 2)
    assert part.tolist() == [0] and cost.tolist() == [one.n, 0]


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


def test_host_pipeline_slices_tile_the_batch():
    """hines_host_pipeline_create (host-only work): the slices are runs of whole cells, tile the batch, and are about
    equal in unknowns when the cells are small against a slice."""
    import morphgen as mg
    import paper_1810_12742_b200 as hb
    m = mg.make_config(3, 0.002)
    for ns in (0, 1, 3, 8, 1000):
        p = hb.HostPipeline(m.parent, m.cell_offsets, nslices=ns)
        s = p.slices
        p.close()
        assert s[0] == 0 and s[-1] == m.n and (np.diff(s) > 0).all()
        assert np.isin(s, m.cell_offsets).all()
        assert len(s) - 1 <= min(ns or 8, m.ncells)
    p = hb.HostPipeline(m.parent, m.cell_offsets, nslices=4)
    sizes = np.diff(p.slices)
    p.close()
    biggest_cell = int(np.diff(m.cell_offsets).max())
    assert len(sizes) == 4 and sizes.max() - sizes.min() <= 2 * biggest_cell
    with pytest.raises(hb.HinesError):
        hb.HostPipeline(m.parent, m.cell_offsets, nslices=-1)
