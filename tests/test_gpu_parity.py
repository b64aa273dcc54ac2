"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Bar (BASELINE.json north_star): per-cell relative max-norm error
<= 1e-10 in fp64; <= 1e-4 in fp32 against the fp64 oracle run on the fp32-rounded inputs
(reading S15)."""
import numpy as np
import pytest

import morphgen as mg
import oracle
from helpers import random_parent

pytestmark = pytest.mark.gpu

TOL = {np.float64: 1e-10, np.float32: 1e-4}


def _gpu_solve(m, d, u, b, dtype=np.float64, inplace=False, **kw):
    import torch
    import paper_1810_12742_b200 as hb
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == np.float64 else hb.F32, **kw)
    dd, du, db = (torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda() for a in (d, u, b))
    x = db if inplace else torch.full_like(db, float("nan"))
    plan.solve(dd, du, db, x)
    torch.cuda.synchronize()
    out = x.cpu().numpy()
    if not inplace:      # inputs are never written
        assert torch.equal(dd.cpu(), torch.from_numpy(np.ascontiguousarray(d, dtype)))
        assert torch.equal(db.cpu(), torch.from_numpy(np.ascontiguousarray(b, dtype)))
    info = plan.info
    plan.close()
    return out, info


def _check(m, d, u, b, dtype=np.float64, **kw):
    x, info = _gpu_solve(m, d, u, b, dtype, **kw)
    dr, ur, br = (np.ascontiguousarray(a, dtype).astype(np.float64) for a in (d, u, b))
    xr = oracle.hines_solve(m.parent, m.cell_offsets, dr, ur, br)
    err = oracle.rel_err(m.cell_offsets, x.astype(np.float64), xr)
    assert np.isfinite(x).all()
    assert err.max() <= TOL[dtype], (err.max(), int(err.argmax()))
    return err.max(), info


SMALL = [(0, 1.0), (1, 0.01), (2, 0.01), (3, 0.003)]


@pytest.mark.parametrize("cfg,scale", SMALL)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_small_configs_default_policy(cfg, scale, dtype):
    m = mg.make_config(cfg, scale)
    d, u, b = mg.system(m)
    _check(m, d, u, b, dtype)


@pytest.mark.parametrize("cfg,scale", SMALL)
def test_small_configs_streaming_path(cfg, scale):
    import paper_1810_12742_b200 as hb
    m = mg.make_config(cfg, scale)
    d, u, b = mg.system(m)
    _, info = _check(m, d, u, b, policy_flags=hb.POLICY_FORCE_STREAM)
    assert info.n_resident_items == 0 and info.n_stream_cells == m.ncells


@pytest.mark.parametrize("kw", [dict(policy_flags=2), dict(policy_flags=4), dict(smem_bytes_per_block=48 * 1024, policy_flags=8),
                                dict(threads_per_block=64), dict(threads_per_block=384, group_smem_bytes=200 * 1024),
                                dict(group_smem_bytes=8 * 1024, stream_threads=32),
                                dict(policy_flags=128), dict(policy_flags=128, max_segment=1023), dict(policy_flags=256),
                                dict(policy_flags=4096), dict(policy_flags=4096, max_segment=1023)])
def test_policy_variants_mixed_paths(kw):
    """Several size classes, resident + streaming in one solve, different block sizes."""
    m = mg.make_config(2, 0.006)
    d, u, b = mg.system(m)
    _, info = _check(m, d, u, b, **kw)
    if kw.get("smem_bytes_per_block"):
        assert info.n_stream_cells > 0 and info.n_resident_items > 0


@pytest.mark.parametrize("kw", [dict(chunk_smem_bytes=40 * 1024), dict(chunk_smem_bytes=24 * 1024, cluster_max=16),
                                dict(chunk_smem_bytes=30 * 1024, cluster_max=2, max_segment=9),
                                dict(chunk_smem_bytes=16 * 1024, cluster_max=16, max_segment=3, threads_per_block=64)])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_cluster_path(kw, dtype):
    """Cells cut into chunks over a thread-block cluster (distributed shared memory), sizes 2..16."""
    m = mg.make_config(2, 0.006)
    d, u, b = mg.system(m)
    _, info = _check(m, d, u, b, dtype, **kw)
    assert info.n_cluster_cells > 0 and info.n_parts > info.n_resident_items


@pytest.mark.parametrize("max_segment", [0, 2, 7, 48, 64, 200, 1023])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_long_cables_segment_targets(max_segment, dtype):
    """Unbranched cables cut into 1..500 segments: odd segment lengths, late-starting lanes, the tight run loop of
    the backward sweep and the turn-around at the root in place of the pointer-jumping rounds."""
    m = mg.make_config(1, 0.002)
    d, u, b = mg.system(m)
    _, info = _check(m, d, u, b, dtype, max_segment=max_segment)
    assert info.n_resident_items > 0 and info.n_stream_cells == 0


def _edge_morphology():
    star = np.array([-1] + [0] * 70, np.int32)            # 70 siblings: hand-off spans tiles (atomic path)
    ps = [np.array([-1], np.int32), star, random_parent(33, 1), np.array([-1], np.int32),
          random_parent(201, 2, .7), star[:40], np.arange(-1, 6, dtype=np.int32),
          random_parent(1001, 3, .97), np.array([-1, 0], np.int32), random_parent(77, 5, .2)]
    if sum(len(p) for p in ps) % 2 == 0:
        ps.append(np.array([-1, 0, 0], np.int32))           # make N odd: the last item ends off a 16-byte boundary
    offs = np.concatenate([[0], np.cumsum([len(p) for p in ps])])
    return mg.Morphology(np.concatenate(ps), offs)          # odd offsets, odd N, non-BFS numbering


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("kw", [{}, dict(policy_flags=1), dict(policy_flags=2), dict(smem_bytes_per_block=8 * 1024)])
def test_edge_cases(dtype, kw):
    m = _edge_morphology()
    assert m.n % 2 == 1
    d, u, b = mg.system(m, seed=11)
    _check(m, d, u, b, dtype, **kw)


def test_in_place_and_nan_poisoned_root_u():
    m = _edge_morphology()
    d, u, b = mg.system(m, seed=12)
    x0, _ = _gpu_solve(m, d, u, b)
    u2 = u.copy(); u2[m.cell_offsets[:-1]] = np.nan         # reading S2: u[root] is never used
    for kw in ({}, dict(policy_flags=1)):
        x1, _ = _gpu_solve(m, d, u2, b, inplace=True, **kw)
        xr = oracle.hines_solve(m.parent, m.cell_offsets, d, u, b)
        assert np.isfinite(x1).all()
        assert oracle.rel_err(m.cell_offsets, x1, xr).max() < 1e-10
    assert np.array_equal(x0, _gpu_solve(m, d, u, b)[0])     # run-to-run deterministic


def test_row_sums_give_ones_on_gpu():
    m = mg.make_config(2, 0.005)
    d, u, _ = mg.system(m)
    b1 = oracle.matvec(m.parent, m.cell_offsets, d, u, np.ones(m.n))
    x, _ = _gpu_solve(m, d, u, b1)
    assert np.abs(x - 1).max() < 1e-13


def test_bad_pointers_rejected():
    import torch
    import paper_1810_12742_b200 as hb
    m = mg.make_config(0)
    plan = hb.Plan(m.parent, m.cell_offsets)
    t = torch.zeros(m.n + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(hb.HinesError) as e:
        plan.solve(t[1:], t[1:], t[1:], t[1:])               # 8-byte aligned only
    assert e.value.status == 1
    with pytest.raises(hb.HinesError):
        plan.solve(t, t, t, t)                               # x aliases d
    big = torch.zeros(4 * m.n + 64, dtype=torch.float64, device="cuda")
    dd, du, db = big[:m.n], big[m.n:2 * m.n], big[2 * m.n:3 * m.n]
    with pytest.raises(hb.HinesError) as e:
        plan.solve(dd, du, db, big[2 * m.n + 2:3 * m.n + 2])  # x overlaps b without being b
    assert e.value.status == 1
    with pytest.raises(hb.HinesError):
        plan.solve(dd, du, db, big[m.n - 2:2 * m.n - 2])      # x overlaps d and u
    plan.solve(dd + 1.0, du, db, db)                          # exactly b: allowed
    torch.cuda.synchronize()


def test_two_live_plans_interleaved():
    """a plan that needs the largest shared memory and a small one, solved in turn (kernel attributes
    are per process, not per plan)."""
    import torch
    import paper_1810_12742_b200 as hb
    ma, mb_ = mg.make_config(2, 0.004), mg.make_config(0)
    pa = hb.Plan(ma.parent, ma.cell_offsets, policy_flags=hb.POLICY_NO_CLUSTER, chunk_smem_bytes=227 * 1024)
    pb = hb.Plan(mb_.parent, mb_.cell_offsets)
    assert pa.table("class_smem_bytes").max() > 150 * 1024 > pb.table("class_smem_bytes").max()
    sa, sb = mg.system(ma), mg.system(mb_)
    ta = [torch.from_numpy(a).cuda() for a in sa]; tb = [torch.from_numpy(a).cuda() for a in sb]
    xa, xb = torch.empty_like(ta[0]), torch.empty_like(tb[0])
    for _ in range(3):
        pa.solve(*ta, xa); pb.solve(*tb, xb)
    torch.cuda.synchronize()
    for m_, s_, x_ in ((ma, sa, xa), (mb_, sb, xb)):
        xr = oracle.hines_solve(m_.parent, m_.cell_offsets, *s_)
        xg = x_.cpu().numpy()
        assert np.isfinite(xg).all() and oracle.rel_err(m_.cell_offsets, xg, xr).max() < 1e-10


@pytest.mark.parametrize("kw", [dict(max_segment=8), dict(max_segment=8, dtype=np.float32), {}])
def test_long_root_branch_with_fork(kw):
    """20,000-compartment root branch with a fork at its end (thousands of reduced nodes on one chain)."""
    n = 20000
    p = np.arange(-1, n + 1, dtype=np.int32)
    p[n + 1] = n - 1
    m = mg.Morphology(p, np.array([0, n + 2], np.int64))
    d, u, b = mg.system(m, seed=3)
    kw = dict(kw); dtype = kw.pop("dtype", np.float64)
    _check(m, d, u, b, dtype, **kw)


@pytest.mark.parametrize("kw", [dict(smem_bytes_per_block=48000, cluster_max=2, split_smem_bytes=20000),
                                dict(smem_bytes_per_block=64000, cluster_max=2, split_smem_bytes=12000, max_segment=9),
                                dict(smem_bytes_per_block=100000, chunk_smem_bytes=30000, cluster_max=3, split_smem_bytes=30000)])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_split_items(kw, dtype):
    """Cells beyond the largest cluster: sub-tree parts backward + export, top part, sub-tree parts again (three launches),
    beside ordinary items in the same solve."""
    m = mg.make_config(2, 0.006)
    d, u, b = mg.system(m)
    _, info = _check(m, d, u, b, dtype, **kw)
    if dtype == np.float64:                                  # (in fp32 the last option set fits its cells into clusters)
        assert info.n_split_cells > 0 and info.n_blocks > info.n_parts


# ---- full BASELINE.json sizes, in the launch configuration bench.py times ----------------------
@pytest.mark.parametrize("cfg,dtype", [(1, np.float64), (2, np.float64), (2, np.float32), (4, np.float64)])
def test_full_size(cfg, dtype):
    m = mg.make_config(cfg, 1.0)
    d, u, b = mg.system(m)
    err, info = _check(m, d, u, b, dtype)
    print(f"cfg{cfg} {np.dtype(dtype).name}: n={m.n} max rel err {err:.3e} resident_items={info.n_resident_items} "
          f"stream_cells={info.n_stream_cells}")


def test_full_size_config3():
    m = mg.make_config(3, 1.0)
    d, u, b = mg.system(m)
    err, info = _check(m, d, u, b)
    print(f"cfg3: n={m.n} max rel err {err:.3e} resident_items={info.n_resident_items} stream_cells={info.n_stream_cells}")


def test_config4_fresh_rhs_steps():
    """Config 4: one very large cell solved for several time steps with a fresh b each step."""
    import torch
    import paper_1810_12742_b200 as hb
    m = mg.make_config(4)
    d, u, _ = mg.system(m)
    plan = hb.Plan(m.parent, m.cell_offsets)
    dd, du = torch.from_numpy(d).cuda(), torch.from_numpy(u).cuda()
    x = torch.empty_like(dd)
    for step in (0, 1, 2, 999):
        b = mg.rhs(m, step=step)
        plan.solve(dd, du, torch.from_numpy(b).cuda(), x)
        xr = oracle.hines_solve(m.parent, m.cell_offsets, d, u, b)
        xg = x.cpu().numpy()
        assert np.isfinite(xg).all()
        assert oracle.rel_err(m.cell_offsets, xg, xr).max() < 1e-10
    plan.close()


# ---- f3: factor once / solve many ----------------------------------------------
def _check_factored(m, d, u, dtype=np.float64, steps=(0, 1, 7), **kw):
    """hines_factor once, hines_solve_rhs per step with a fresh b, against the oracle's two-function split of
    Listing 2 (oracle.hines_factor / hines_solve_rhs) on the inputs as the GPU sees them."""
    import torch
    import paper_1810_12742_b200 as hb
    flags = kw.pop("policy_flags", 0) | hb.POLICY_FACTORED
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == np.float64 else hb.F32, policy_flags=flags, **kw)
    dd, du = (torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda() for a in (d, u))
    dr, ur = (np.ascontiguousarray(a, dtype).astype(np.float64) for a in (d, u))
    dw, f = oracle.hines_factor(m.parent, m.cell_offsets, dr, ur)
    plan.factor(dd, du)
    dd.fill_(float("nan")); du.fill_(float("nan"))             # the factors are the plan's: d, u are not read again
    worst = 0.0
    for step in steps:
        b = mg.rhs(m, step=step)
        db = torch.from_numpy(np.ascontiguousarray(b, dtype)).cuda()
        x = torch.full_like(db, float("nan"))
        plan.solve_rhs(db, x)
        torch.cuda.synchronize()
        xg = x.cpu().numpy().astype(np.float64)
        br = np.ascontiguousarray(b, dtype).astype(np.float64)
        xr = oracle.hines_solve_rhs(m.parent, m.cell_offsets, dw, f, ur, br)
        assert np.isfinite(xg).all()
        err = oracle.rel_err(m.cell_offsets, xg, xr).max()
        assert err <= TOL[dtype], (step, err)
        worst = max(worst, err)
        plan.solve_rhs(db, db)                                  # in place
        torch.cuda.synchronize()
        assert torch.equal(db, x)
    info = plan.info
    plan.close()
    return worst, info


@pytest.mark.parametrize("cfg,scale", SMALL)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_factored_small_configs(cfg, scale, dtype):
    m = mg.make_config(cfg, scale)
    d, u, _ = mg.system(m)
    _check_factored(m, d, u, dtype)


@pytest.mark.parametrize("kw", [dict(chunk_smem_bytes=40 * 1024), dict(chunk_smem_bytes=24 * 1024, cluster_max=16, max_segment=9),
                                dict(smem_bytes_per_block=80000, cluster_max=2, split_smem_bytes=26000),
                                dict(policy_flags=2), dict(policy_flags=128), dict(policy_flags=4096)])
def test_factored_clusters_split_items_policies(kw):
    m = mg.make_config(2, 0.006)
    d, u, _ = mg.system(m)
    _check_factored(m, d, u, **kw)
    me = _edge_morphology()
    d, u, _ = mg.system(me, seed=11)
    _check_factored(me, d, u, **{k: v for k, v in kw.items() if k == "policy_flags"})


def test_factored_needs_the_flag_and_the_factor_call():
    import torch
    import paper_1810_12742_b200 as hb
    m = mg.make_config(0)
    d, u, b = (torch.from_numpy(a).cuda() for a in mg.system(m))
    plan = hb.Plan(m.parent, m.cell_offsets)
    with pytest.raises(hb.HinesError) as e:
        plan.factor(d, u)
    assert e.value.status == 5
    plan = hb.Plan(m.parent, m.cell_offsets, policy_flags=hb.POLICY_FACTORED)
    with pytest.raises(hb.HinesError) as e:
        plan.solve_rhs(b, torch.empty_like(b))
    assert e.value.status == 1
    x = torch.empty_like(b)                                     # a factored plan still serves the full solve
    plan.solve(d, u, b, x)
    torch.cuda.synchronize()
    xr = oracle.hines_solve(m.parent, m.cell_offsets, *mg.system(m))
    assert oracle.rel_err(m.cell_offsets, x.cpu().numpy(), xr).max() < 1e-10


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_factored_full_size(cfg):
    m = mg.make_config(cfg, 1.0)
    d, u, _ = mg.system(m)
    err, info = _check_factored(m, d, u, steps=(0, 999) if cfg == 4 else (1,))
    print(f"cfg{cfg} factored: n={m.n} max rel err {err:.3e} split_cells={info.n_split_cells} cluster_cells={info.n_cluster_cells}")


# ---- f2, tree re-rooting: badly rooted cells solved as given and after hines_reroot, the permutation
#      carried through load and store by hines_gather / hines_scatter; both against the oracle on the cells as given ----
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_rerooted_cells_through_gather_and_scatter(dtype):
    import torch
    import paper_1810_12742_b200 as hb
    from helpers import rooted_at
    hd = hb.F64 if dtype == np.float64 else hb.F32
    m0 = mg.make_config(2, 0.004)
    d0, u0, b0 = mg.system(m0)
    # the same cells rooted at a leaf (their last compartment): the badly balanced input
    parent, perm0, usrc0 = rooted_at(m0.parent, m0.cell_offsets, lambda c, n: n - 1)
    d, u, b = d0[perm0], u0[usrc0], b0[perm0]
    dr, ur, br = (np.ascontiguousarray(a, dtype).astype(np.float64) for a in (d, u, b))
    xr = oracle.hines_solve(parent, m0.cell_offsets, dr, ur, br)
    rr = hb.reroot(parent, m0.cell_offsets)
    assert (rr["depth_after"] < rr["depth_before"]).all()
    dd, du, db = (torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda() for a in (d, u, b))
    perm, usrc = torch.from_numpy(rr["perm"]).cuda(), torch.from_numpy(rr["u_src"]).cuda()
    d2, u2, b2 = torch.full_like(dd, float("nan")), torch.full_like(dd, float("nan")), torch.full_like(dd, float("nan"))
    hb.gather(d2, dd, perm, hd); hb.gather(u2, du, usrc, hd); hb.gather(b2, db, perm, hd)
    torch.cuda.synchronize()
    assert torch.equal(d2, dd[perm]) and torch.equal(u2, du[usrc]) and torch.equal(b2, db[perm])      # bit-exact index work
    before, after = hb.Plan(parent, m0.cell_offsets, dtype=hd), hb.Plan(rr["new_parent"], m0.cell_offsets, dtype=hd)
    try:
        assert after.info.max_levels < before.info.max_levels
        x_given = torch.full_like(dd, float("nan"))
        before.solve(dd, du, db, x_given)
        x2, x = torch.full_like(dd, float("nan")), torch.full_like(dd, float("nan"))
        after.solve(d2, u2, b2, x2)
        hb.scatter(x, x2, perm, hd)
        torch.cuda.synchronize()
        for xs in (x_given, x):
            xs = xs.cpu().numpy().astype(np.float64)
            assert np.isfinite(xs).all()
            assert oracle.rel_err(m0.cell_offsets, xs, xr).max() <= TOL[dtype]
    finally:
        before.close(); after.close()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("pinned", [True, False])
def test_host_pipeline_matches_oracle(dtype, pinned):
    """hines_host_pipeline_solve: host buffers in and out, slices overlapped; twice in a row with a fresh right-hand side."""
    import torch
    import paper_1810_12742_b200 as hb
    m = mg.make_config(3, 0.004)
    d, u, _ = mg.coefficients(m, mg.rng.BASE_SEED)
    pipe = hb.HostPipeline(m.parent, m.cell_offsets, dtype=hb.F64 if dtype == np.float64 else hb.F32, nslices=5)
    try:
        assert len(pipe.slices) == 6
        for step in range(2):
            b = mg.rhs(m, mg.rng.BASE_SEED, step)
            bufs = [np.ascontiguousarray(a, dtype) for a in (d, u, b)] + [np.full(m.n, np.nan, dtype)]
            if pinned:
                bufs = [torch.from_numpy(a).pin_memory() for a in bufs]
            pipe.solve(*bufs)
            x = (bufs[3].numpy() if pinned else bufs[3]).astype(np.float64)
            dr, ur, br = (np.ascontiguousarray(a, dtype).astype(np.float64) for a in (d, u, b))
            xr = oracle.hines_solve(m.parent, m.cell_offsets, dr, ur, br)
            assert np.isfinite(x).all()
            assert oracle.rel_err(m.cell_offsets, x, xr).max() <= TOL[dtype]
    finally:
        pipe.close()
