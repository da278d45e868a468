"""GPU parity of the importer (PAPER.md:430 / :219): cuth_import_csr condenses a CSR matrix into the
matrix object bit for bit, validates it like the oracle's entry-by-entry checker, and the solver runs on it."""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
from gpu_util import grid_from_workload, to_dev
from import_faults import faults

pytestmark = pytest.mark.gpu

CASES = [
    dict(cfg=1, nx=2, ny=2, nz=2, n_hot=0),
    dict(cfg=1, nx=7, ny=2, nz=5, n_hot=1),
    dict(cfg=3, nx=37, ny=29, nz=16, n_hot=8),     # per-cell lognormal kappa
    dict(cfg=5, nx=48, ny=40, nz=16, n_hot=8),     # C/dt on the diagonal: every layer has a non-zero row sum
    dict(cfg=4, nx=130, ny=67, nz=8, n_hot=6),
    dict(cfg=6, nx=45, ny=38, nz=10, n_hot=6),
]


def _csr_dev(A):
    import torch
    return (torch.from_numpy(A.rowptr).cuda(), torch.from_numpy(A.col).cuda(), torch.from_numpy(A.val).cuda())


def _exact_rowsums(w):
    s = np.zeros(w.nz)
    s[-1] += w.h_top * (w.dx * w.dy)
    if w.cvol is not None and w.dt > 0:
        s += np.asarray(w.cvol) * ((w.dx * w.dy) * np.asarray(w.dz)) / w.dt
    return s


def _shuffle_rows(A, seed):
    """Same matrix with the entries of every row in a different order."""
    rng = np.random.default_rng(seed)
    col, val = A.col.copy(), A.val.copy()
    for i in range(A.n):
        a, b = int(A.rowptr[i]), int(A.rowptr[i + 1])
        p = rng.permutation(b - a)
        col[a:b] = A.col[a:b][p]
        val[a:b] = A.val[a:b][p]
    return O.CSR(A.n, A.rowptr.copy(), col, val)


@pytest.mark.parametrize("kw", CASES + [dict(cfg=2)])
@pytest.mark.parametrize("given_rowsums", [False, True])
def test_import_is_bit_exact(kw, given_rowsums):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    vals_o, ptr_o, off_o = O.csr_to_dia(A, w.nx, w.ny, w.nz)
    g = grid_from_workload(w)
    A_sh = _shuffle_rows(A, 7) if w.n <= 100000 else A
    M = cu.DiaMatrix(g, csr=_csr_dev(A_sh), rowsum_layer=_exact_rowsums(w) if given_rowsums else None)
    rep = M.import_report
    assert (rep.off_stencil, rep.asymmetric_rows, rep.bad_diagonal, rep.duplicates, rep.positive_offdiag) == (0,) * 5
    assert rep.mixed_ok == 1 and rep.max_rowsum_dev <= 1e-9
    vals, vals32, inv, ptr, off = M.view()
    assert ptr == ptr_o.tolist() and off == off_o.tolist()
    assert np.array_equal(vals.cpu().numpy().view(np.uint64), vals_o.view(np.uint64))
    assert np.array_equal(vals32.cpu().numpy().view(np.uint32), vals_o.astype(np.float32).view(np.uint32))
    assert np.array_equal(inv.cpu().numpy(), 1.0 / vals_o[:w.n])
    # everything the solver kernels read besides the per-layer table is byte-identical to what the builder writes
    B = cu.DiaMatrix(g)
    lay_end = 512 + 256 * (((4 * w.nz + 4) * 8 + 255) // 256)
    al = lambda v: (v + 255) // 256 * 256                    # section alignment of the matrix object
    e, n = int(ptr[4]), w.n
    o_h16 = al(al(al(lay_end + 8 * e) + 4 * e) + 8 * n)      # after A1, A2, 1/D0
    o_f32a = o_h16 + 3 * al(2 * n)
    o_f64a = o_f32a + 3 * al(4 * n)
    for k in range(3):                          # A3 (fp16, scaled) and the aligned per-diagonal copies of A2 and of A1
        a, b, c = o_h16 + k * al(2 * n), o_f32a + k * al(4 * n), o_f64a + k * al(8 * n)
        assert bool((M.buf[a:a + 2 * n] == B.buf[a:a + 2 * n]).all())
        assert bool((M.buf[b:b + 4 * n] == B.buf[b:b + 4 * n]).all())
        assert bool((M.buf[c:c + 8 * n] == B.buf[c:c + 8 * n]).all())
        # the aligned fp64 copy of diagonal k+1 is the packed diagonal followed by a zero tail
        dk = M.buf[c:c + 8 * n].view(np_to_torch_f64()).cpu().numpy()
        lk = int(ptr[k + 2] - ptr[k + 1])
        assert np.array_equal(dk[:lk].view(np.uint64), vals_o[int(ptr[k + 1]):int(ptr[k + 2])].view(np.uint64))
        assert not dk[lk:].any()
    o_dinv32 = o_f64a + 3 * al(8 * n)                        # fp32(1/D0): the early-stage preconditioner of the fused path
    assert bool((M.buf[o_dinv32:o_dinv32 + 4 * n] == B.buf[o_dinv32:o_dinv32 + 4 * n]).all())
    import torch
    d32 = M.buf[o_dinv32:o_dinv32 + 4 * n].view(torch.float32).cpu().numpy()
    assert np.array_equal(d32.view(np.uint32), (1.0 / vals_o[:n]).astype(np.float32).view(np.uint32))
    assert o_dinv32 + al(4 * n) == M.buf.numel()
    sc = slice(512 + 32 * w.nz, 512 + 32 * w.nz + 24)        # |entry|max bits, fp16 scale, 1/scale
    assert bool((M.buf[sc] == B.buf[sc]).all())
    s_imp = M.buf[512 + 8 * w.nz: 512 + 16 * w.nz].view(np_to_torch_f64()).cpu().numpy()
    s_bld = B.buf[512 + 8 * w.nz: 512 + 16 * w.nz].view(np_to_torch_f64()).cpu().numpy()
    if given_rowsums:
        assert np.array_equal(s_imp, s_bld)
    else:
        assert np.abs(s_imp - s_bld).max() <= 1e-9 * vals_o[:w.n].min()


def np_to_torch_f64():
    import torch
    return torch.float64


@pytest.mark.parametrize("kw", CASES)
def test_solve_on_imported_matrix(kw):
    """FP64 and MIXED solves on the imported object meet the same bars as on the built one (north_star)."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    ref = O.pcg(A, w.power, rtol=1e-10)
    assert ref.status == 0
    g = grid_from_workload(w)
    M = cu.DiaMatrix(g, csr=_csr_dev(A))
    B = cu.DiaMatrix(g)
    for precision, bar in ((cu.FP64, 1e-6 * np.abs(ref.x).max()), (cu.MIXED, 1e-4)):
        xs = []
        for mat in (M, B):
            S = cu.Solver(mat, cu.Opts(precision=precision, rtol=1e-8, true_resid_period=w.true_resid_period))
            x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
            S.solve(to_dev(w.power), x)
            res = S.result()
            assert res.status == 0
            xs.append(x.cpu().numpy())
            S.close()
        assert np.abs(xs[0] - ref.x).max() <= bar
        r = w.power - O.spmv(A, xs[0])
        assert np.linalg.norm(r) <= 1e-8 * np.linalg.norm(w.power)
        if precision == cu.FP64:
            assert np.array_equal(xs[0], xs[1])        # same bytes in, same kernels: identical iterates


def test_validation_counts_match_the_oracle():
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=3, nx=12, ny=9, nz=5, n_hot=2)
    A = O.assemble_workload(w)
    g = grid_from_workload(w)
    import torch
    buf = torch.empty(cu.cuth_dia_bytes(g), dtype=torch.uint8, device="cuda")
    for name, Af in faults(A, w.nx, w.ny, w.nz).items():
        want = O.stencil7_report(Af, w.nx, w.ny, w.nz)
        rc, rep = cu.cuth_import_csr(g, *_csr_dev(Af), buf, check=False)
        got = dict(off_stencil=rep.off_stencil, asymmetric_rows=rep.asymmetric_rows, bad_diagonal=rep.bad_diagonal,
                   duplicates=rep.duplicates, positive_offdiag=rep.positive_offdiag)
        assert got == {k: want[k] for k in got}, name
        healthy = name == "explicit_zero_off_stencil"
        assert rc == (0 if healthy else -8), name


def test_non_layered_row_sums_are_fp64_only():
    """A diagonal shift that varies from cell to cell keeps A SPD but leaves no per-layer row sum: the import
    succeeds, MIXED is refused ON THE DEVICE (the object's own header says so: status CUTH_SOLVE_FP64_ONLY, x untouched
    -- also for a byte copy of the object at another address, which a host-side table keyed by address would miss), and the
    FP64 solve matches the oracle on the same matrix."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=3, nx=20, ny=14, nz=6, n_hot=3)
    A = O.assemble_workload(w)
    rows = np.repeat(np.arange(A.n), np.diff(A.rowptr))
    dq = np.flatnonzero(A.col == rows)
    v = A.val.copy()
    v[dq] *= 1.0 + 0.05 * W.uniform01(w.seed, 77, np.arange(A.n))
    Ap = O.CSR(A.n, A.rowptr, A.col, v)
    want = O.stencil7_report(Ap, w.nx, w.ny, w.nz)
    assert want["mixed_ok"] == 0
    g = grid_from_workload(w)
    M = cu.DiaMatrix(g, csr=_csr_dev(Ap))
    assert M.import_report.mixed_ok == 0
    assert M.import_report.max_rowsum_dev == pytest.approx(want["max_rowsum_dev"], rel=1e-6)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S = cu.Solver(M, cu.Opts(precision=cu.MIXED))
    x.fill_(3.25)
    S.solve(to_dev(w.power), x)
    r = S.result()
    assert r.status == cu.SOLVE_FP64_ONLY and r.iterations == 0 and bool((x == 3.25).all())
    buf2 = M.buf.clone()                                   # the same object at another address
    res2 = torch.zeros(64, dtype=torch.uint8, device="cuda")
    cu.cuth_pcg_solve(buf2, g, S.opts, to_dev(w.power), x, S.work, res2)
    torch.cuda.synchronize()
    assert int(res2[:4].view(torch.int32).item()) == cu.SOLVE_FP64_ONLY and bool((x == 3.25).all())
    SB = cu.BatchSolver(M, 2, cu.Opts(precision=cu.MIXED))
    xb = torch.full((2, w.n), 3.25, dtype=torch.float64, device="cuda")
    SB.solve(torch.stack([to_dev(w.power)] * 2), xb)
    assert [q.status for q in SB.results()] == [cu.SOLVE_FP64_ONLY] * 2 and bool((xb == 3.25).all())
    assert not np.isfinite(M.spmv(to_dev(w.power), cu.MIXED).cpu().numpy()).any()   # s(z) = NaN: fails loudly
    x.zero_()
    S = cu.Solver(M, cu.Opts(precision=cu.FP64))
    S.solve(to_dev(w.power), x)
    assert S.result().status == 0
    ref = O.pcg(Ap, w.power, rtol=1e-10)
    assert np.abs(x.cpu().numpy() - ref.x).max() <= 1e-6 * np.abs(ref.x).max()
    # a supplied per-layer table that the matrix contradicts is an error
    rc, rep = cu.cuth_import_csr(g, *_csr_dev(Ap), M.buf, rowsum_layer=_exact_rowsums(w), check=False)
    assert rc == -8 and rep.mixed_ok == 0
    # and the same buffer rebuilt by cuth_build_dia is a normal matrix again
    cu.cuth_build_dia(g, M.buf)
    S = cu.Solver(M, cu.Opts(precision=cu.MIXED))
    S.solve(to_dev(w.power), x.zero_())
    assert S.result().status == 0


def test_import_rejects_a_malformed_rowptr_before_reading_through_it():
    """a rowptr that is not a row pointer (not starting at 0, decreasing, pointing beyond the arrays, absurd row
    lengths) must end in CUTH_ERR_STRUCTURE with `bad_rowptr` counted -- not in out-of-bounds reads of col / val."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=1, nx=6, ny=5, nz=4, n_hot=1)
    A = O.assemble_workload(w)
    g = grid_from_workload(w)
    rp, col, val = _csr_dev(A)
    buf = torch.empty(cu.cuth_dia_bytes(g), dtype=torch.uint8, device="cuda")
    nnz = int(A.rowptr[-1])

    def bad(rowptr_np, expect, nnz_arg=None):
        rc, rep = cu.cuth_import_csr(g, torch.from_numpy(rowptr_np).cuda(), col, val, buf, check=False, nnz=nnz_arg)
        assert rc == -8 and rep.bad_rowptr == expect and rep.mixed_ok == 0, (rc, rep.bad_rowptr, expect)

    r = A.rowptr.copy(); r[0] = 1
    bad(r, 1)                                                    # does not start at 0
    r = A.rowptr.copy(); r[10] = r[9] - 1
    bad(r, 1)                                                    # decreasing: row 9 ends before it starts (row 10 just gets longer)
    r = A.rowptr.copy(); r[-1] = nnz + 1000
    bad(r, 1, nnz_arg=nnz)                                       # last row runs beyond the arrays (caught because nnz is known)
    r = A.rowptr.copy(); r[5:] += 1 << 40
    bad(r, 1, nnz_arg=-1)                                        # nnz unknown: row 4 would have 2^40 entries
    bad(r, w.n - 4)                                              # nnz known: rows 4 .. n-1 all end beyond the arrays
    r = A.rowptr.copy(); r[3] = -7
    bad(r, 2)                                                    # negative pointer: rows 2 and 3
    rc, rep = cu.cuth_import_csr(g, rp, col, val, buf, check=False)          # and the real thing still imports
    assert rc == 0 and rep.bad_rowptr == 0 and rep.mixed_ok == 1


def test_import_argument_errors():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=1, nx=4, ny=3, nz=2, n_hot=1)
    A = O.assemble_workload(w)
    g = grid_from_workload(w)
    rp, col, val = _csr_dev(A)
    buf = torch.empty(cu.cuth_dia_bytes(g), dtype=torch.uint8, device="cuda")
    L = cu.load_library()
    import ctypes as C
    from paper_2606_17850_b200.binding import cuth_import_report_t
    rep = cuth_import_report_t()
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    p = lambda t: C.c_void_p(t.data_ptr())
    assert L.cuth_import_csr(g.ref(), None, p(col), p(val), None, p(buf), buf.numel(), C.byref(rep), st) == -1
    assert L.cuth_import_csr(g.ref(), p(rp), p(col), p(val), None, p(buf), buf.numel() - 1, C.byref(rep), st) == -4
    assert L.cuth_import_csr(g.ref(), p(rp), p(col), p(val), None, C.c_void_p(buf.data_ptr() + 8), buf.numel(),
                             C.byref(rep), st) == -5
    bad = np.full(w.nz, -1.0)
    assert L.cuth_import_csr(g.ref(), p(rp), p(col), p(val), bad.ctypes.data_as(C.c_void_p), p(buf), buf.numel(),
                             C.byref(rep), st) == -3
    # an imported matrix is a steady operator for this library
    wt = W.make_workload(cfg=5, nx=8, ny=6, nz=4, n_hot=2)
    gt = grid_from_workload(wt)
    M = cu.DiaMatrix(gt, csr=_csr_dev(O.assemble_workload(wt)))
    S = cu.Solver(M, cu.Opts())
    T = torch.full((wt.n,), 1.5, dtype=torch.float64, device="cuda")
    S.step(to_dev(wt.power), T)
    r = S.result()
    assert r.status == cu.SOLVE_NOT_TRANSIENT and r.iterations == 0 and bool((T == 1.5).all())


def _coo_dev(A, seed=None):
    """The CSR matrix as (row, col, val) int32 / int32 / float64 device arrays, entries shuffled when seed is given."""
    import torch
    rows = np.repeat(np.arange(A.n, dtype=np.int32), np.diff(A.rowptr))
    cols, vals = A.col.astype(np.int32), A.val
    if seed is not None:
        p = np.random.default_rng(seed).permutation(rows.size)
        rows, cols, vals = rows[p], cols[p], vals[p]
    return (torch.from_numpy(np.ascontiguousarray(rows)).cuda(), torch.from_numpy(np.ascontiguousarray(cols)).cuda(),
            torch.from_numpy(np.ascontiguousarray(vals)).cuda())


@pytest.mark.parametrize("kw", CASES + [dict(cfg=2)])
def test_import_coo_is_bit_exact(kw):
    """cuth_import_coo on the shuffled entries writes byte for byte the object cuth_import_csr writes."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    vals_o, _, _ = O.csr_to_dia(A, w.nx, w.ny, w.nz)
    g = grid_from_workload(w)
    M = cu.DiaMatrix(g, csr=_csr_dev(A))
    buf = torch.empty_like(M.buf)
    rep = cu.cuth_import_coo(g, *_coo_dev(A, seed=11), buf)
    assert (rep.off_stencil, rep.asymmetric_rows, rep.bad_diagonal, rep.duplicates, rep.positive_offdiag) == (0,) * 5
    assert rep.mixed_ok == 1 and rep.max_rowsum_dev == M.import_report.max_rowsum_dev
    v, _, _, ptr, _ = cu.cuth_dia_view(buf, g)
    e = ptr[4]
    got = buf[v - buf.data_ptr(): v - buf.data_ptr() + 8 * e].view(torch.float64).cpu().numpy()
    assert np.array_equal(got.view(np.uint64), vals_o.view(np.uint64))
    lay_end = 512 + 256 * (((4 * w.nz + 4) * 8 + 255) // 256)
    al = lambda q: (q + 255) // 256 * 256
    n = w.n
    sections = [(512 + 8 * w.nz, 8 * w.nz), (512 + 32 * w.nz, 24), (lay_end, 8 * e), (al(lay_end + 8 * e), 4 * e),
                (al(al(lay_end + 8 * e) + 4 * e), 8 * n)]                  # s(z) | fp16 scale | A1 | A2 | 1/D0
    o_h16 = al(al(al(lay_end + 8 * e) + 4 * e) + 8 * n)
    o_f32a = o_h16 + 3 * al(2 * n)
    sections += [(o_h16 + k * al(2 * n), 2 * n) for k in range(3)] + [(o_f32a + k * al(4 * n), 4 * n) for k in range(3)]
    for a, nb in sections:
        assert bool((buf[a:a + nb] == M.buf[a:a + nb]).all()), a
    # and it solves: MIXED on the COO-imported object
    x = torch.zeros(n, dtype=torch.float64, device="cuda")
    opts = cu.Opts(precision=cu.MIXED, true_resid_period=w.true_resid_period)
    work = torch.empty(cu.cuth_workspace_bytes(g, opts), dtype=torch.uint8, device="cuda")
    res = torch.zeros(64, dtype=torch.uint8, device="cuda")
    cu.cuth_pcg_solve(buf, g, opts, to_dev(w.power), x, work, res)
    torch.cuda.synchronize()
    cu.cuth_release_workspace(work)
    assert int(res[:4].view(torch.int32).item()) == 0
    r = w.power - O.spmv(A, x.cpu().numpy())
    assert np.linalg.norm(r) <= 1e-8 * np.linalg.norm(w.power)


def test_coo_validation_counts_match_the_oracle():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=3, nx=12, ny=9, nz=5, n_hot=2)
    A = O.assemble_workload(w)
    g = grid_from_workload(w)
    buf = torch.empty(cu.cuth_dia_bytes(g), dtype=torch.uint8, device="cuda")
    for name, Af in faults(A, w.nx, w.ny, w.nz).items():
        want = O.stencil7_report(Af, w.nx, w.ny, w.nz)
        rc, rep = cu.cuth_import_coo(g, *_coo_dev(Af, seed=5), buf, check=False)
        got = dict(off_stencil=rep.off_stencil, asymmetric_rows=rep.asymmetric_rows, bad_diagonal=rep.bad_diagonal,
                   duplicates=rep.duplicates, positive_offdiag=rep.positive_offdiag)
        if name == "duplicate":        # which copy of a repeated coordinate is kept is unspecified: only its count is
            assert got["duplicates"] == want["duplicates"] == 1
        else:
            assert got == {k: want[k] for k in got}, name
        assert rc == (0 if name == "explicit_zero_off_stencil" else -8), name
    # a lower triangle that is missing altogether: every row with a lower neighbour is asymmetric
    rows = np.repeat(np.arange(A.n), np.diff(A.rowptr))
    keep = A.col >= rows
    up = (torch.from_numpy(rows[keep].astype(np.int32)).cuda(), torch.from_numpy(A.col[keep].astype(np.int32)).cuda(),
          torch.from_numpy(A.val[keep]).cuda())
    rc, rep = cu.cuth_import_coo(g, *up, buf, check=False)
    assert rc == -8 and rep.asymmetric_rows == A.n - 1 and rep.off_stencil == 0
