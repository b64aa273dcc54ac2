"""hines_solve_static -- the entry point that allocates nothing (scratch in a static __device__ array inside the library)
-- against the existing path (hines_solve with an uploaded plan), on two calls in a row, within the tolerances of the
other GPU tests.  Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

import morphgen as mg

pytestmark = pytest.mark.gpu

TOL = {np.float64: 1e-10, np.float32: 1e-4}      # the bar of tests/test_gpu_parity.py


def _rel_err(cell_offsets, x, xr):
    """Per-cell relative max-norm error (the measure of the parity tests), computed here: no oracle needed, both sides
    are GPU results."""
    err = np.zeros(len(cell_offsets) - 1)
    for c in range(len(err)):
        lo, hi = cell_offsets[c], cell_offsets[c + 1]
        err[c] = np.abs(x[lo:hi] - xr[lo:hi]).max() / max(np.abs(xr[lo:hi]).max(), 1e-300)
    return err


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("cfg,scale", [(0, 1.0), (2, 0.004)])
def test_static_entry_matches_plan_path_twice(cfg, scale, dtype):
    import torch
    import paper_1810_12742_b200 as hb
    hd = hb.F64 if dtype == np.float64 else hb.F32
    m = mg.make_config(cfg, scale)
    d, u, _ = mg.coefficients(m, mg.rng.BASE_SEED)
    assert m.n * np.dtype(dtype).itemsize <= hb.STATIC_SCRATCH_BYTES
    parent = torch.from_numpy(np.ascontiguousarray(m.parent, np.int32)).cuda()
    offs = torch.from_numpy(np.ascontiguousarray(m.cell_offsets, np.int64)).cuda()
    dd, du = (torch.from_numpy(np.ascontiguousarray(a, dtype)).cuda() for a in (d, u))
    plan = hb.Plan(m.parent, m.cell_offsets, dtype=hd)
    try:
        for step in range(2):                          # two calls in a row: the second meets the first one's scratch
            b = mg.rhs(m, mg.rng.BASE_SEED, step)
            db = torch.from_numpy(np.ascontiguousarray(b, dtype)).cuda()
            x_ref = torch.full_like(db, float("nan"))
            plan.solve(dd, du, db, x_ref)
            x = torch.full_like(db, float("nan"))
            hb.solve_static(parent, offs, dd, du, db, x, dtype=hd)
            torch.cuda.synchronize()
            xs, xr = x.cpu().numpy().astype(np.float64), x_ref.cpu().numpy().astype(np.float64)
            assert np.isfinite(xs).all() and np.isfinite(xr).all()
            err = _rel_err(m.cell_offsets, xs, xr)
            assert err.max() <= TOL[dtype], (step, err.max(), int(err.argmax()))
            # inputs are never written
            assert torch.equal(db.cpu(), torch.from_numpy(np.ascontiguousarray(b, dtype)))
            assert torch.equal(dd.cpu(), torch.from_numpy(np.ascontiguousarray(d, dtype)))
        # in place (x == b) gives the same bits as out of place
        xb = db.clone()
        hb.solve_static(parent, offs, dd, du, xb, xb, dtype=hd)
        torch.cuda.synchronize()
        assert torch.equal(xb, x)
    finally:
        plan.close()


def test_static_entry_rejects_sizes_beyond_the_array():
    import torch
    import paper_1810_12742_b200 as hb
    m = mg.make_config(0, 1.0)
    d, u, b = mg.system(m)
    parent = torch.from_numpy(np.ascontiguousarray(m.parent, np.int32)).cuda()
    offs = torch.from_numpy(np.ascontiguousarray(m.cell_offsets, np.int64)).cuda()
    dd, du, db = (torch.from_numpy(a).cuda() for a in (d, u, b))
    x = torch.empty_like(db)
    lib = hb.load_library()
    too_many = hb.STATIC_SCRATCH_BYTES // 8 + 1        # rejected before anything is touched
    st = lib.hines_solve_static(parent.data_ptr(), offs.data_ptr(), m.ncells, too_many, dd.data_ptr(), du.data_ptr(),
                                db.data_ptr(), x.data_ptr(), hb.F64, None)
    assert st == 5                                     # HINES_ERR_UNSUPPORTED
    msg = lib.hines_last_error().decode()
    assert "exceeds the static scratch array" in msg and str(hb.STATIC_SCRATCH_BYTES) in msg
    st = lib.hines_solve_static(None, offs.data_ptr(), m.ncells, m.n, dd.data_ptr(), du.data_ptr(), db.data_ptr(),
                                x.data_ptr(), hb.F64, None)
    assert st == 1                                     # HINES_ERR_INVALID_ARG
