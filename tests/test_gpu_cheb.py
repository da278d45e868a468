"""GPU parity of the Chebyshev path: Lanczos bounds, one preconditioner apply
(Alg. 3) and the PCG solve, against the CPU oracle, in both grid traversals."""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
from oracle import stored_operators as SO
from gpu_util import grid_from_workload, to_dev

pytestmark = pytest.mark.gpu

CASES = [
    dict(cfg=1, nx=7, ny=5, nz=4, n_hot=1),
    dict(cfg=1),
    dict(cfg=3, nx=37, ny=29, nz=16, n_hot=8),
    dict(cfg=5, nx=48, ny=40, nz=16, n_hot=8),
    dict(cfg=4, nx=130, ny=67, nz=8, n_hot=6),
    dict(cfg=6, nx=45, ny=38, nz=10, n_hot=6),     # paper-like anisotropic stack
    dict(cfg=4, nx=136, ny=67, nz=8, n_hot=6),     # nx % 8 == 0: three x-tiles of the TMA two-pass kernel, ragged in x and y
    dict(cfg=1, nx=8, ny=4, nz=2, n_hot=1),        # two planes only: every plane of the march is a peeled one
]


@pytest.fixture(params=["flat", "flat-pairs", "flat-pairs-ldg", "zmarch", "zmarch-x1"], autouse=True)
def traversal(request):
    import paper_2606_17850_b200 as cu
    cu.set_default_tuning(traversal=1 if request.param.startswith("flat") else 2)
    # "flat", "zmarch-x1" = one pass per kernel; "flat-pairs", "zmarch" = two passes per kernel (operands by TMA
    # when nx % 4 == 0 (fp16: % 8), by ordinary loads otherwise); "flat-pairs-ldg" = two passes, never TMA
    cu.set_default_tuning(cheb_fusion={"flat": 1, "flat-pairs": 2, "flat-pairs-ldg": 3, "zmarch": 2, "zmarch-x1": 1}[request.param],
                          k1_variant=1 if request.param == "zmarch-x1" else 2)   # 2: two columns per thread when nx is even
    yield request.param
    cu.set_default_tuning(traversal=0, k1_variant=0, cheb_fusion=0)


# fp32 apply against Alg. 3 evaluated in fp64 on the SAME stored operator, max-abs over max-abs: 29 passes of fp32
# arithmetic (unit roundoff 6e-8) with the amplification of the three-term recurrence; measured <= 1.9e-6 on every case
# and kernel schedule on B200 (printed by the tests with -s), bar set five times above.
FP32_APPLY_TOL = 1e-5


def _row_sums(w):
    s = np.zeros((w.nz, w.nx * w.ny))
    s[w.nz - 1] += w.h_top * w.dx * w.dy
    if w.transient:
        s += (w.cvol * (w.dx * w.dy * w.dz) / w.dt)[:, None]
    return s.reshape(-1)


def _rhs(w):
    return w.power if not w.transient else O.transient_rhs(w, w.power, np.zeros(w.n))


def _setup(w, prec, steps=20, degree=30, storage=0):
    import paper_2606_17850_b200 as cu
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.Solver(M, cu.Opts(precision=prec, rtol=1e-8, true_resid_period=w.true_resid_period))
    b = _rhs(w)
    lo, hi, gersh = S.setup_chebyshev(to_dev(b), lanczos_steps=steps, degree=degree, storage=storage)
    return M, S, b, lo, hi, gersh


@pytest.mark.parametrize("kw", CASES)
def test_lanczos_bounds_vs_oracle(kw):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    steps = 12
    M, S, b, lo, hi, gersh = _setup(w, cu.FP64, steps=steps)
    a, bt = O.lanczos(A, b, steps)
    lo_o, hi_o = O.ritz_extremes(a, bt)
    assert hi == pytest.approx(hi_o, rel=1e-6)
    assert lo == pytest.approx(lo_o, rel=1e-4)
    rowsum = np.abs(A.to_scipy()).sum(axis=1).max()
    assert gersh == pytest.approx(rowsum, rel=1e-12)
    assert S.opts.cheb_lmin == lo and S.opts.cheb_lmax == min(1.05 * hi, gersh)


@pytest.mark.parametrize("kw", CASES)
@pytest.mark.parametrize("degree", [3, 4, 30])
def test_cheb_apply_fp64_vs_oracle(kw, degree):
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    M, S, b, lo, hi, gersh = _setup(w, cu.FP64, degree=degree)
    r = W.normal01(w.seed, 50, 51, np.arange(w.n)) * 1e-7
    z = torch.empty(w.n, dtype=torch.float64, device="cuda")
    S.cheb_apply(to_dev(r), z)
    ref = O.cheb_apply(A, r, S.opts.cheb_lmin, S.opts.cheb_lmax, degree)
    assert np.abs(z.cpu().numpy() - ref).max() <= 1e-10 * np.abs(ref).max()


@pytest.mark.parametrize("kw", CASES)
def test_cheb_apply_fp32_close_to_oracle(kw):
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    M, S, b, lo, hi, gersh = _setup(w, cu.MIXED)
    r = W.normal01(w.seed, 50, 51, np.arange(w.n)) * 1e-7
    z = torch.empty(w.n, dtype=torch.float64, device="cuda")
    S.cheb_apply(to_dev(r), z)
    # ELEMENT-WISE reference: Alg. 3 in fp64 on the operator the kernel really multiplies by -- the fp32-rounded
    # off-diagonals in difference form (oracle/stored_operators.py).  What is left is the fp32 rounding of the vector
    # arithmetic over 29 passes; a wrong rim cell, a mis-scaled entry or a dropped term on one plane is O(1) of |z|.
    ref = O.cheb_apply(SO.fp32_difference_operator(A, _row_sums(w)), r, S.opts.cheb_lmin, S.opts.cheb_lmax, 30)
    zg = z.cpu().numpy()
    print("fp32 apply: max-abs / |z|inf =", np.abs(zg - ref).max() / np.abs(ref).max())
    assert np.abs(zg - ref).max() <= FP32_APPLY_TOL * np.abs(ref).max()
    exact = O.cheb_apply(A, r, S.opts.cheb_lmin, S.opts.cheb_lmax, 30)
    assert np.linalg.norm(zg - exact) <= 2e-3 * np.linalg.norm(exact)          # and still a preconditioner for A itself


@pytest.mark.parametrize("kw", CASES)
def test_pcg_cheb_fp64_vs_oracle(kw):
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    M, S, b, lo, hi, gersh = _setup(w, cu.FP64)
    ref = O.pcg_cheb(A, b, S.opts.cheb_lmin, S.opts.cheb_lmax, 30)
    assert ref.status == 0
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(to_dev(b), x)
    res = S.result()
    xh = x.cpu().numpy()
    assert res.status == 0, res
    assert np.linalg.norm(b - O.spmv(A, xh)) <= 1e-8 * np.linalg.norm(b)
    assert np.abs(xh - ref.x).max() <= 1e-6 * np.abs(ref.x).max()
    assert abs(res.iterations - ref.iterations) <= max(3, 0.1 * ref.iterations)
    jac = O.pcg(A, b)
    assert np.abs(xh - jac.x).max() <= 1e-6 * np.abs(jac.x).max()      # same x whatever the preconditioner


@pytest.mark.parametrize("kw", CASES)
def test_pcg_cheb_mixed_vs_oracle(kw):
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    M, S, b, lo, hi, gersh = _setup(w, cu.MIXED)
    ref = O.pcg(A, b)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(to_dev(b), x)
    res = S.result()
    xh = x.cpu().numpy()
    assert res.status == 0, res
    assert np.linalg.norm(b - O.spmv(A, xh)) <= 1e-8 * np.linalg.norm(b)
    assert np.abs(xh - ref.x).max() <= 1e-4
    if w.n >= 8192:
        assert res.iterations < ref.iterations / 2                      # far fewer outer iterations than Jacobi


@pytest.mark.parametrize("kw", CASES)
def test_cheb_fp16_matrix_apply_and_solve(kw):
    """A3: half-precision off-diagonals (times a power-of-two scale), promoted to fp32 on load (Alg. 4's
    arithmetic decoupling).  The apply is a 2^-11-accurate copy of the same operator;
    the solve must still meet both parity bars, the outer loop and the true residual being fp64."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    M, S, b, lo, hi, gersh = _setup(w, cu.MIXED, storage=cu.CHEB_A3_FP16)
    r = W.normal01(w.seed, 50, 51, np.arange(w.n)) * 1e-7
    z = torch.empty(w.n, dtype=torch.float64, device="cuda")
    S.cheb_apply(to_dev(r), z)
    # element-wise against Alg. 3 in fp64 on the fp16-stored operator (scale S, difference form): pins the scale, the
    # zero tails and every rim cell of the kernels that read A3
    ref = O.cheb_apply(SO.fp16_difference_operator(A, _row_sums(w)), r, S.opts.cheb_lmin, S.opts.cheb_lmax, 30)
    zg = z.cpu().numpy()
    print("fp16 apply: max-abs / |z|inf =", np.abs(zg - ref).max() / np.abs(ref).max())
    assert np.abs(zg - ref).max() <= FP32_APPLY_TOL * np.abs(ref).max()
    exact = O.cheb_apply(A, r, S.opts.cheb_lmin, S.opts.cheb_lmax, 30)
    assert np.linalg.norm(zg - exact) <= 2e-2 * np.linalg.norm(exact)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(to_dev(b), x)
    res = S.result()
    xh = x.cpu().numpy()
    assert res.status == 0, res
    assert np.linalg.norm(b - O.spmv(A, xh)) <= 1e-8 * np.linalg.norm(b)
    assert np.abs(xh - O.pcg(A, b).x).max() <= 1e-4


@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=3, nx=37, ny=29, nz=16, n_hot=8), dict(cfg=5, nx=48, ny=40, nz=16, n_hot=8)])
@pytest.mark.parametrize("traversal", ["flat-pairs"], indirect=True)
def test_lanczos_fp32_variant_vs_reference_and_solve(kw, traversal):
    """Lanczos in FP32 with the fixed-FP32 SpMV on A2 (`cuth_tuning_t.lanczos_fp32`).  Against the
    step-by-step fp32 reference (oracle/ablation.py, whose fp64 instance reproduces oracle_lanczos): the spectral interval
    agrees to a few per cent (unconverged Ritz values move with the summation order); the interval serves the
    preconditioner as well as the fp64 one (R-C5): same outer iteration count to within 15 %, both bars met."""
    import torch
    import paper_2606_17850_b200 as cu
    from oracle import ablation as AB
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    b = _rhs(w)
    M = cu.DiaMatrix(grid_from_workload(w))
    out = {}
    for f32 in (0, 1):
        S = cu.Solver(M, cu.Opts(precision=cu.MIXED, rtol=1e-8, true_resid_period=w.true_resid_period,
                                 tuning=cu.Tuning(lanczos_fp32=f32)))
        lo, hi, gersh = S.setup_chebyshev(to_dev(b), lanczos_steps=20, degree=30)
        x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        S.solve(to_dev(b), x)
        r = S.result()
        assert r.status == 0 and np.linalg.norm(b - O.spmv(A, x.cpu().numpy())) <= 1e-8 * np.linalg.norm(b)
        out[f32] = (lo, hi, r.iterations)
        S.close()
    a32, b32 = AB.lanczos_fixed(A, b, 20, dtype=np.float32)
    lo_o, hi_o = O.ritz_extremes(a32, b32)
    assert out[1][1] == pytest.approx(hi_o, rel=0.02) and out[1][0] == pytest.approx(lo_o, rel=0.1)
    assert out[1][1] == pytest.approx(out[0][1], rel=0.02)
    assert abs(out[1][2] - out[0][2]) <= max(3, 0.15 * out[0][2])


def test_lanczos_invariant_subspace_on_a_tiny_grid():
    """N = 8 < requested Lanczos steps: the Krylov space is exhausted (beta_j -> 0); the bounds must still be
    the exact extreme eigenvalues and the Chebyshev solve must work."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1, nx=2, ny=2, nz=2, n_hot=0)
    A = O.assemble_workload(w)
    lam = np.linalg.eigvalsh(A.to_scipy().toarray())
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.Solver(M, cu.Opts(precision=cu.FP64))
    v0 = W.uniform01(7, 70, np.arange(w.n)) + 0.1          # generic start vector (b is constant per layer here)
    lo, hi, gersh = S.setup_chebyshev(to_dev(v0), lanczos_steps=20, degree=5)
    assert lam[0] * (1 - 1e-6) <= lo <= lam[-1] and hi == pytest.approx(lam[-1], rel=1e-6)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(to_dev(w.power), x)
    res = S.result()
    assert res.status == 0
    xs = np.linalg.solve(A.to_scipy().toarray(), w.power)
    assert np.abs(x.cpu().numpy() - xs).max() <= 1e-6 * np.abs(xs).max()


def test_cheb_bad_interval_rejected_or_reported():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1, nx=8, ny=6, nz=4, n_hot=1)
    M = cu.DiaMatrix(grid_from_workload(w))
    bad = cu.Opts(preconditioner=cu.PRECOND_CHEBYSHEV, cheb_degree=30, cheb_lmin=1.0, cheb_lmax=0.5)
    S = cu.Solver(M, bad)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    with pytest.raises(cu.CuthError) as e:
        S.solve(to_dev(w.power), x)
    assert e.value.code == -3
    S2 = cu.Solver(M, cu.Opts(preconditioner=cu.PRECOND_CHEBYSHEV, cheb_degree=2, cheb_lmin=1e-6, cheb_lmax=1e-3))
    with pytest.raises(cu.CuthError):
        S2.solve(to_dev(w.power), x)


SHAPES = [(4, 2, 2), (8, 6, 3), (12, 9, 5), (64, 8, 2), (60, 6, 4), (68, 10, 4), (124, 13, 3), (128, 7, 9),
          (200, 31, 6), (256, 64, 16)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("degree", [5, 6, 30])
@pytest.mark.parametrize("storage", ["fp32", "fp16"])
@pytest.mark.parametrize("traversal", ["flat"], indirect=True)       # the test sets the schedule itself: once
def test_cheb_apply_kernel_variants_agree(shape, degree, storage, traversal):
    """The same polynomial through the three kernel schedules of the fp32 apply -- one pass per kernel, two
    passes per kernel with ordinary loads, two passes per kernel with TMA-staged operands (taken when nx % 4 == 0,
    fp16: % 8; regions of 8 and of 16 rows) -- on shapes below, at and above one 60 x 6 region, with per-cell conductivities: every row runs
    the same arithmetic, so the results agree to fp32 rounding of the order of operations."""
    import torch
    import paper_2606_17850_b200 as cu
    nx, ny, nz = shape
    w = W.make_workload(3, nx=nx, ny=ny, nz=nz, n_hot=2)
    M, S, b, lo, hi, gersh = _setup(w, cu.MIXED, steps=min(20, w.n - 1), degree=degree,
                                    storage=cu.CHEB_A3_FP16 if storage == "fp16" else cu.CHEB_DEFAULT)
    r = W.normal01(w.seed, 52, 53, np.arange(w.n)) * 1e-7
    out = {}
    for mode, rows in ((1, 0), (3, 0), (2, 8), (2, 16)):      # rows: region height of the TMA kernel
        S.opts.tuning.cheb_fusion = mode                       # per-call tuning (cuth_tuning_t)
        S.opts.tuning.pair_rows = rows
        z = torch.full((w.n,), float("nan"), dtype=torch.float64, device="cuda")
        S.cheb_apply(to_dev(r), z)
        out[(mode, rows)] = z.cpu().numpy()
    ref = out[(1, 0)]
    assert np.isfinite(ref).all()
    scale = np.abs(ref).max()
    for key in ((3, 0), (2, 8), (2, 16)):
        assert np.abs(out[key] - ref).max() <= 2e-5 * scale, (key, shape)


@pytest.mark.parametrize("traversal", ["flat-pairs"], indirect=True)
def test_graph_cache_follows_plane_shape_and_matrix(traversal):
    """The TMA two-pass nodes carry tensor maps baked into the cached graph of a workspace.  Re-using the SAME
    workspace and the SAME matrix buffer for another grid with the same N (planes transposed: identical buffer
    sizes, identical block counts are possible) must rebuild the graph, not reuse stale maps."""
    import torch
    import paper_2606_17850_b200 as cu
    shapes = [(120, 12, 6), (12, 120, 6), (120, 12, 6)]
    copts = cu.Opts(cu.MIXED, 1e-8, 20000, 20, cu.PRECOND_CHEBYSHEV, 30, 1e-3, 1.0)
    wls = [W.make_workload(3, nx=nx, ny=ny, nz=nz, n_hot=3) for (nx, ny, nz) in shapes]
    grids = [grid_from_workload(w) for w in wls]
    buf = torch.empty(max(cu.cuth_dia_bytes(g) for g in grids), dtype=torch.uint8, device="cuda")
    work = torch.empty(max(cu.cuth_workspace_bytes(g, copts) for g in grids), dtype=torch.uint8, device="cuda")
    res = torch.zeros(64, dtype=torch.uint8, device="cuda")
    for (nx, ny, nz), w, g in zip(shapes, wls, grids):
        cu.cuth_build_dia(g, buf)
        b = to_dev(w.power)
        lo, hi, gersh, rlo, rhi = cu.cuth_lanczos_bounds(buf, g, b, 20, work)
        opts = cu.Opts(cu.MIXED, 1e-8, 20000, 20, cu.PRECOND_CHEBYSHEV, 30, rlo, rhi)
        x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        cu.cuth_pcg_solve(buf, g, opts, b, x, work, res)
        torch.cuda.synchronize()
        A = O.assemble_workload(w)
        xg = x.cpu().numpy()
        rel = np.linalg.norm(w.power - O.spmv(A, xg)) / np.linalg.norm(w.power)
        assert rel <= 1e-8, (nx, ny, nz, rel)
    cu.cuth_release_workspace(work)


@pytest.mark.parametrize("traversal", ["flat-pairs"], indirect=True)
def test_graph_cache_follows_the_workspace_layout(traversal):
    """A transient matrix keeps b in the workspace, which moves the Chebyshev buffers N doubles later -- and their
    addresses are baked into the tensor maps of the cached TMA nodes.  Steady, then transient, then steady again on
    the SAME workspace and the SAME matrix buffer (same N, same plane): every solve must meet the bar."""
    import torch
    import paper_2606_17850_b200 as cu
    ws = W.make_workload(2, nx=48, ny=40, nz=16, n_hot=8)
    wt = W.make_workload(5, nx=48, ny=40, nz=16, n_hot=8)
    gs, gt = grid_from_workload(ws), grid_from_workload(wt)
    copts = cu.Opts(cu.MIXED, 1e-8, 20000, 5, cu.PRECOND_CHEBYSHEV, 30, 1e-3, 1.0)
    buf = torch.empty(max(cu.cuth_dia_bytes(gs), cu.cuth_dia_bytes(gt)), dtype=torch.uint8, device="cuda")
    work = torch.empty(max(cu.cuth_workspace_bytes(gs, copts), cu.cuth_workspace_bytes(gt, copts)), dtype=torch.uint8,
                       device="cuda")
    res = torch.zeros(64, dtype=torch.uint8, device="cuda")
    for w, g in ((ws, gs), (wt, gt), (ws, gs)):
        cu.cuth_build_dia(g, buf)
        A = O.assemble_workload(w)
        b_np = _rhs(w)
        b = to_dev(b_np)
        lo, hi, gersh, rlo, rhi = cu.cuth_lanczos_bounds(buf, g, b, 20, work)
        opts = cu.Opts(cu.MIXED, 1e-8, 20000, 5, cu.PRECOND_CHEBYSHEV, 30, rlo, rhi)
        x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        cu.cuth_pcg_solve(buf, g, opts, b, x, work, res)
        torch.cuda.synchronize()
        assert int(res[:4].view(torch.int32).item()) == 0, w.name
        rel = np.linalg.norm(b_np - O.spmv(A, x.cpu().numpy())) / np.linalg.norm(b_np)
        assert rel <= 1e-8, (w.name, rel)
    cu.cuth_release_workspace(work)
