"""cuth_residual_noalloc (include/cuth.h): the one entry point that needs no workspace and allocates nothing -- its
reduction scratch is a file-scope device array.  Checked against the EXISTING path (cuth_spmv through the C ABI, then
t = b - y and the two norms in fp64 with torch) on two calls in a row that share the scratch: the second call runs on a
smaller grid than the first, so stale partial sums of the first call sit right behind the slots it uses.
Named test_zz_* so that pytest collects it last (the suite runs with pytest -x)."""
import numpy as np
import pytest

import workloads as W
from gpu_util import grid_from_workload, to_dev

pytestmark = pytest.mark.gpu


def _existing_path(cu, torch, M, b, x):
    y = M.spmv(x, cu.FP64)                        # cuth_spmv_tuned -> k_spmv_only<OP_FP64>
    t = b - y
    return t, float((t * t).sum()), float((b * b).sum())


def test_residual_noalloc_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    import paper_2606_17850_b200 as cu
    out = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    cases = [dict(cfg=4, nx=130, ny=67, nz=8, n_hot=6),      # 69 680 rows: 9 CTAs, ragged tail
             dict(cfg=3, nx=37, ny=29, nz=16, n_hot=8),      # 17 168 rows: 3 CTAs -- slots 3..8 hold the first call's sums
             dict(cfg=1, nx=2, ny=2, nz=2, n_hot=0)]         # the smallest grid the ABI accepts
    prepared = []
    for kw in cases:
        w = W.make_workload(**kw)
        M = cu.DiaMatrix(grid_from_workload(w))
        b = to_dev(w.power)
        x = to_dev(W.normal01(w.seed, 70, 71, np.arange(w.n)) * 1e-2 + 3.0)
        t = torch.full((w.n,), float("nan"), dtype=torch.float64, device="cuda")
        prepared.append((w, M, b, x, t))
    torch.cuda.synchronize()
    for rep in range(2):                                         # the whole sequence twice: six calls back to back
        for w, M, b, x, t in prepared:
            t.fill_(float("nan")); out.fill_(float("nan"))
            cu.cuth_residual_noalloc(M.buf, M.grid, b, x, out, t=t)
            t_ref, tt_ref, bb_ref = _existing_path(cu, torch, M, b, x)
            o = out.cpu().numpy()
            # same operator, same order of operations per row as the fp64 SpMV kernel: t agrees to the last bits of y
            scale = float(t_ref.abs().max())
            assert float((t - t_ref).abs().max()) <= 1e-12 * scale
            assert o[0] == pytest.approx(tt_ref, rel=1e-12) and o[1] == pytest.approx(bb_ref, rel=1e-12)
            assert o[2] == pytest.approx(np.sqrt(tt_ref / bb_ref), rel=1e-12) and o[3] == 0.0
            # norms only (t_D = NULL), bit-identical to the call before: fixed-order sums, no stale scratch
            out2 = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
            cu.cuth_residual_noalloc(M.buf, M.grid, b, x, out2)
            assert np.array_equal(out2.cpu().numpy().view(np.uint64), o.view(np.uint64))
    # zero right-hand side: relative residual reported as 0
    w, M, b, x, t = prepared[1]
    cu.cuth_residual_noalloc(M.buf, M.grid, torch.zeros_like(b), torch.zeros_like(x), out)
    assert out.cpu().numpy().tolist() == [0.0, 0.0, 0.0, 0.0]


def test_residual_noalloc_agrees_with_a_solve_and_rejects_what_it_cannot_serve():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1)
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.Solver(M, cu.Opts(precision=cu.FP64, rtol=1e-8))
    b = to_dev(w.power)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(b, x)
    r = S.result()
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    cu.cuth_residual_noalloc(M.buf, M.grid, b, x, out)
    assert r.status == 0 and float(out[2]) == pytest.approx(r.rel_resid_true, rel=1e-6) and float(out[2]) <= 1e-8
    S.close()
    # beyond the stated maximum: refused on the host, before anything is launched, with a message that says why
    assert cu.cuth_noalloc_max_rows() == 1 << 24
    big = cu.Grid(4096, 4096, 2, 1e-6, 1e-6, np.full(2, 1e-6), None, 1e4)          # 33.5 M rows
    out.fill_(7.0)
    with pytest.raises(cu.CuthError) as e:
        cu.cuth_residual_noalloc(M.buf, big, b, x, out)
    assert e.value.code == -4 and "maximum of 16777216 rows" in str(e.value)
    torch.cuda.synchronize()
    assert out.cpu().numpy().tolist() == [7.0] * 4
    exact = cu.Grid(1024, 1024, 16, 1e-6, 1e-6, np.full(16, 1e-6), None, 1e4)      # exactly the maximum: accepted by the size check
    assert cu.cuth_residual_noalloc(None, exact, b, x, out, check=False) == -1      # (NULL matrix is the next check)
    assert cu.cuth_residual_noalloc(M.buf, M.grid, b, x, out, t=x, check=False) == -3   # t must not alias x
