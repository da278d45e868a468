"""GPU parity of the batched solve: nrhs right-hand sides on one matrix, each by its
own Alg. 1 recurrence inside one persistent kernel.  Every x_s is compared with the oracle's solve of (A, b_s)."""
import ctypes as C

import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
from gpu_util import grid_from_workload, to_dev
from paper_2606_17850_b200.binding import cuth_result_t

pytestmark = pytest.mark.gpu


@pytest.fixture(params=["auto", "lockstep"], autouse=True)
def home(request):
    """"auto": grids that fit one thread-block cluster run one cluster-resident solve per right-hand side (round 2), the
    others the lock-step persistent kernel; "lockstep": the lock-step kernel (k_pcg_batch) everywhere."""
    import paper_2606_17850_b200 as cu
    cu.set_default_tuning(loop_mode=2 if request.param == "lockstep" else 0)
    yield request.param
    cu.set_default_tuning(loop_mode=0)


GRIDS = [
    dict(cfg=1, nx=2, ny=2, nz=2, n_hot=0),
    dict(cfg=1, nx=7, ny=2, nz=5, n_hot=1),
    dict(cfg=1),                                   # BASELINE configs[0]
    dict(cfg=3, nx=37, ny=29, nz=16, n_hot=8),     # per-cell lognormal kappa
    dict(cfg=4, nx=130, ny=67, nz=8, n_hot=6),     # several row tiles + ragged tail
    dict(cfg=6, nx=45, ny=38, nz=10, n_hot=6),
]


def rhs_set(w, nrhs):
    """Seeded right-hand sides of different difficulty: the workload's own power map, modulated copies, a single
    hot cell, and (last, when nrhs >= 3) the zero vector."""
    idx = np.arange(w.n)
    B = np.empty((nrhs, w.n))
    for s in range(nrhs):
        if s == 0:
            B[s] = w.power
        elif s % 3 == 1:
            B[s] = w.power * (0.25 + 1.5 * W.uniform01(w.seed, 100 + s, idx))
        elif s % 3 == 2:
            B[s] = 0.0
            B[s, (7919 * s) % w.n] = np.abs(w.power).max()
        else:
            B[s] = np.abs(W.normal01(w.seed, 200 + s, 300 + s, idx)) * np.abs(w.power).mean()
    if nrhs >= 3:
        B[-1] = 0.0
    return B


def _run(w, B, X0=None, precond=1, rtol=1e-8, max_iters=200000, precision=0, period=20):
    import torch
    import paper_2606_17850_b200 as cu
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.BatchSolver(M, B.shape[0], cu.Opts(precision=precision, rtol=rtol, max_iters=max_iters, preconditioner=precond,
                                              true_resid_period=period))
    x = torch.zeros(B.shape, dtype=torch.float64, device="cuda") if X0 is None else to_dev(X0)
    S.solve(to_dev(B), x)
    return x.cpu().numpy(), S.results(), M


@pytest.mark.parametrize("kw", GRIDS)
@pytest.mark.parametrize("nrhs", [1, 3, 4, 7, 32])
def test_batch_vs_oracle(kw, nrhs):
    w = W.make_workload(**kw)
    if nrhs == 32 and w.n > 20000:
        pytest.skip("32 oracle solves of this grid: covered by nrhs = 7")
    A = O.assemble_workload(w)
    B = rhs_set(w, nrhs)
    X, res, _ = _run(w, B)
    for s in range(nrhs):
        assert res[s].status == 0, s
        if not B[s].any():
            assert not X[s].any() and res[s].iterations == 0
            continue
        ref = O.pcg(A, B[s], rtol=1e-8)
        assert ref.status == 0
        assert np.abs(X[s] - ref.x).max() <= 1e-6 * np.abs(ref.x).max(), s
        r = B[s] - O.spmv(A, X[s])
        assert np.linalg.norm(r) <= 1e-8 * np.linalg.norm(B[s]), s
        assert abs(res[s].iterations - ref.iterations) <= max(5, 0.05 * ref.iterations), (s, res[s].iterations, ref.iterations)
        assert res[s].rel_resid_true == pytest.approx(np.linalg.norm(r) / np.linalg.norm(B[s]), rel=1e-3, abs=1e-10)


@pytest.mark.parametrize("kw", GRIDS[1:])
@pytest.mark.parametrize("nrhs", [2, 6])
def test_batch_mixed_vs_oracle_and_single_policy(kw, nrhs):
    """MIXED: north_star's bars per right-hand side (<= 1e-4 K, oracle-CSR true residual <= 1e-8), and every right-hand
    side takes the stage decisions a single MIXED solve of it takes (same criterion; iteration of the switch and
    iteration count up to the effect of the summation order on a threshold test: one true-residual period)."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    B = rhs_set(w, nrhs)
    T = w.true_resid_period
    X, res, M = _run(w, B, precision=cu.MIXED, period=T)
    S1 = cu.Solver(M, cu.Opts(precision=cu.MIXED, true_resid_period=T))
    for s in range(nrhs):
        assert res[s].status == 0, s
        if not B[s].any():
            continue
        ref = O.pcg(A, B[s], rtol=1e-10)
        assert np.abs(X[s] - ref.x).max() <= 1e-4, s
        r = B[s] - O.spmv(A, X[s])
        assert np.linalg.norm(r) <= 1e-8 * np.linalg.norm(B[s]), s
        x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        S1.solve(to_dev(B[s]), x)
        r1 = S1.result()
        assert res[s].promotions == r1.promotions == 1
        assert res[s].switch_reason == r1.switch_reason
        assert abs(res[s].switch_iteration - r1.switch_iteration) <= T
        assert abs(res[s].iterations - r1.iterations) <= max(3, T)
        assert abs(res[s].true_resid_evals - r1.true_resid_evals) <= 2


def test_batch_matches_single_solves():
    """Same kernels' arithmetic per row: the batch and nrhs single solves agree far below the parity bar, with the same
    iteration counts up to the effect of the summation order on the stopping test."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=3, nx=37, ny=29, nz=16, n_hot=8)
    B = rhs_set(w, 6)
    X, res, M = _run(w, B)
    S1 = cu.Solver(M, cu.Opts(precision=cu.FP64))
    for s in range(6):
        x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
        S1.solve(to_dev(B[s]), x)
        r1 = S1.result()
        assert r1.status == 0 and abs(r1.iterations - res[s].iterations) <= 2
        if B[s].any():
            assert np.abs(x.cpu().numpy() - X[s]).max() <= 1e-7 * np.abs(X[s]).max()


def test_batch_warm_start_and_no_preconditioner():
    w = W.make_workload(cfg=1, nx=12, ny=9, nz=5, n_hot=2)
    A = O.assemble_workload(w)
    B = rhs_set(w, 5)
    refs = [O.pcg(A, B[s], rtol=1e-12).x for s in range(5)]
    X0 = np.zeros_like(B)
    X0[1] = refs[1]                    # already solved: 0 iterations
    X0[2] = 0.5 * refs[2]
    X, res, _ = _run(w, B, X0=X0)
    assert res[1].iterations == 0 and res[1].status == 0 and np.array_equal(X[1], X0[1])
    for s in range(4):
        assert np.abs(X[s] - refs[s]).max() <= 1e-6 * np.abs(refs[s]).max()
    Xn, resn, _ = _run(w, B, precond=0)
    for s in range(4):
        ref = O.pcg(A, B[s], rtol=1e-8, precond=0)
        assert resn[s].status == 0 and abs(resn[s].iterations - ref.iterations) <= max(5, 0.05 * ref.iterations)
        assert np.abs(Xn[s] - refs[s]).max() <= 1e-6 * np.abs(refs[s]).max()


def test_batch_iteration_cap_is_per_right_hand_side():
    w = W.make_workload(cfg=3, nx=37, ny=29, nz=16, n_hot=8)
    B = rhs_set(w, 4)
    X, res, _ = _run(w, B, max_iters=10)
    assert [r.status for r in res] == [1, 1, 1, 0] and [r.iterations for r in res] == [10, 10, 10, 0]
    assert all(r.rel_resid_true > 1e-8 for r in res[:3])


def test_batch_argument_errors():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(cfg=1, nx=4, ny=3, nz=2, n_hot=1)
    g = grid_from_workload(w)
    M = cu.DiaMatrix(g)
    assert cu.cuth_batch_workspace_bytes(g, 0) == 0 and cu.cuth_batch_workspace_bytes(g, 33) == 0
    S = cu.BatchSolver(M, 2)
    b = torch.ones(2, w.n, dtype=torch.float64, device="cuda")
    x = torch.zeros_like(b)

    def code(opts, nrhs=2, work=None):
        work = S.work if work is None else work
        with pytest.raises(cu.CuthError) as e:
            cu.cuth_pcg_solve_batch(M.buf, g, opts, nrhs, b, x, work, S.result_dev)
        return e.value.code

    assert code(cu.Opts(preconditioner=cu.PRECOND_CHEBYSHEV, cheb_lmin=1.0, cheb_lmax=2.0)) == -3
    assert code(cu.Opts(), nrhs=0) == -3 and code(cu.Opts(), nrhs=33) == -3
    assert code(cu.Opts(), work=S.work[:S.work.numel() - 256]) == -4


@pytest.mark.parametrize("kw", [dict(cfg=1, nx=7, ny=5, nz=3, n_hot=1), dict(cfg=4, nx=130, ny=67, nz=8, n_hot=6)])
@pytest.mark.parametrize("nrhs", [3, 9])
def test_batch_and_import_no_out_of_bounds_canaries(kw, nrhs):
    """Same stand-in for memcheck as test_no_out_of_bounds_canaries (compute-sanitizer is closed on this pool), for
    the two calls added last: every caller-owned buffer (CSR arrays, matrix object, b, x, workspace, result records) is
    carved with exactly the size the ABI asks for out of a NaN-filled arena; guard words must survive bitwise, and the
    results must be bit-identical to the run on ordinary allocations."""
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    g = grid_from_workload(w)
    A = O.assemble_workload(w)
    B = rhs_set(w, nrhs)
    nanbits = torch.tensor([float("nan")], dtype=torch.float64, device="cuda").view(torch.int64)

    def run(guarded):
        pad = 4096 if guarded else 0
        arenas, bufs = {}, {}

        def carve(name, nbytes):
            nb8 = (nbytes + 7) // 8 * 8
            arena = torch.full(((nb8 + 2 * pad) // 8,), float("nan"), dtype=torch.float64, device="cuda").view(torch.uint8)
            arenas[name] = (arena, nb8)
            bufs[name] = arena[pad:pad + nbytes]

        carve("rowptr", A.rowptr.nbytes); carve("col", A.col.nbytes); carve("val", A.val.nbytes)
        carve("dia", cu.cuth_dia_bytes(g)); carve("b", B.nbytes); carve("x", B.nbytes)
        carve("work", cu.cuth_batch_workspace_bytes(g, nrhs)); carve("res", nrhs * C.sizeof(cuth_result_t))
        bufs["rowptr"].view(torch.int64).copy_(torch.from_numpy(A.rowptr))
        bufs["col"].view(torch.int32).copy_(torch.from_numpy(A.col))
        bufs["val"].view(torch.float64).copy_(torch.from_numpy(A.val))
        rep = cu.cuth_import_csr(g, bufs["rowptr"].view(torch.int64), bufs["col"].view(torch.int32),
                                 bufs["val"].view(torch.float64), bufs["dia"])
        assert rep.mixed_ok == 1
        bufs["b"].view(torch.float64).copy_(to_dev(B).reshape(-1))
        x = bufs["x"].view(torch.float64)
        x.zero_()
        cu.cuth_pcg_solve_batch(bufs["dia"], g, cu.Opts(), nrhs, bufs["b"].view(torch.float64), x, bufs["work"], bufs["res"])
        torch.cuda.synchronize()
        if guarded:
            for name, (arena, nb8) in arenas.items():
                assert bool((arena[:pad].view(torch.int64) == nanbits).all()), f"guard below {name} overwritten"
                assert bool((arena[pad + nb8:].view(torch.int64) == nanbits).all()), f"guard above {name} overwritten"
        return x.clone().cpu().numpy(), bufs["res"].view(torch.int32).cpu().numpy().copy()

    x0, r0 = run(False)
    x1, r1 = run(True)
    assert np.array_equal(r0, r1) and np.array_equal(x0.view(np.uint64), x1.view(np.uint64))
    assert all(r0[(C.sizeof(cuth_result_t) // 4) * s] == 0 for s in range(nrhs))
