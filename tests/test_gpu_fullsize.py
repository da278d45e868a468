"""GPU parity at BASELINE.json's FULL sizes (cfg 3, 4, 5), in the launch configuration bench.py times.

A full CPU PCG on these grids takes minutes to hours, so the CUDA result is checked through quantities the
oracle (or a pin that shares no code with either side) can compute at this size:
  * the true fp64 relative residual of the GPU's x evaluated with the ORACLE's independently assembled CSR,
  * global energy balance (eq. (4)/(5) summed over all cells),
  * x >= 0 for b >= 0 (M-matrix),
  * for layered conductivity (cfg 4, 5) the separable direct solve (tests/direct_solve.py) as truth for
    every unknown; for cfg 5 additionally the oracle PCG on the first steps.
cfg 3 (per-cell lognormal kappa) has no closed form at full size: invariants only.
"""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
from direct_solve import solve_layered
from gpu_util import grid_from_workload, to_dev

pytestmark = pytest.mark.gpu


def _solve(w, prec, b=None, chebyshev=False):
    import torch
    import paper_2606_17850_b200 as cu
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.Solver(M, cu.Opts(precision=prec, rtol=1e-8, true_resid_period=w.true_resid_period))
    bd = to_dev(w.power if b is None else b)
    if chebyshev:
        S.setup_chebyshev(bd, lanczos_steps=40, degree=30)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(bd, x)
    res = S.result()
    xh = x.cpu().numpy()
    S.close()
    del S, M, x
    torch.cuda.empty_cache()
    return xh, res


def _check_invariants(w, A, b, x, res):
    assert res.status == 0, res
    rel = np.linalg.norm(b - O.spmv(A, x)) / np.linalg.norm(b)
    assert rel <= 1e-8, rel
    assert abs(rel - res.rel_resid_true) <= 1e-3 * rel + 1e-13        # device-reported value agrees
    assert np.all(x >= 0.0)
    top = x.reshape(w.nz, -1)[w.nz - 1]
    out = (w.h_top * w.dx * w.dy) * top.sum()
    assert out == pytest.approx(b.sum(), rel=1e-6)                   # injected power = heat through the top


@pytest.mark.parametrize("mode", ["fp64", "mixed"])
def test_cfg3_full_size(mode):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(3)
    A = O.assemble_workload(w)
    x, res = _solve(w, cu.FP64 if mode == "fp64" else cu.MIXED)
    _check_invariants(w, A, w.power, x, res)
    if mode == "fp64":
        assert res.promotions == 0
        # sampled rows: (A x)_i recomputed one by one from the oracle CSR equals b_i to the residual level
        idx = (W.uniform01(w.seed, 40, np.arange(64)) * w.n).astype(np.int64)
        for i in idx:
            s = 0.0
            for k in range(A.rowptr[i], A.rowptr[i + 1]):
                s += A.val[k] * x[A.col[k]]
            assert abs(s - w.power[i]) <= 1e-6 * np.abs(A.val[A.rowptr[i]:A.rowptr[i + 1]]).max() * x.max()


def test_cfg3_full_size_chebyshev_mixed():
    import paper_2606_17850_b200 as cu
    w = W.make_workload(3)
    A = O.assemble_workload(w)
    x, res = _solve(w, cu.MIXED, chebyshev=True)
    _check_invariants(w, A, w.power, x, res)
    assert res.iterations < 1000                 # Jacobi needs 4499 (Table VII: 44-107 vs 647-1593)
    xj, _ = _solve(w, cu.FP64)
    assert np.abs(x - xj).max() <= 1e-4          # same temperatures as the Jacobi fp64 solve


@pytest.mark.parametrize("mode", ["fp64", "mixed", "chebyshev-mixed"])
def test_cfg4_full_size(mode):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(4)
    x, res = _solve(w, cu.FP64 if mode == "fp64" else cu.MIXED, chebyshev=mode.startswith("chebyshev"))
    assert res.status == 0, res
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    err = np.abs(x - xd).max()
    if mode == "fp64":
        assert err <= 1e-6 * np.abs(xd).max(), err
    else:
        assert err <= 1e-4, err
    del xd
    A = O.assemble_workload(w)
    _check_invariants(w, A, w.power, x, res)


@pytest.mark.parametrize("mode", ["fp64", "mixed", "chebyshev-fp64", "chebyshev-mixed"])
def test_cfg6_paperlike_stack_full_size(mode):
    """cfg 6 (the paper's ten layer thicknesses; 256x256x10): layered, so the separable direct
    solve is the truth for every unknown."""
    import paper_2606_17850_b200 as cu
    w = W.make_workload(6)
    A = O.assemble_workload(w)
    x, res = _solve(w, cu.FP64 if mode.endswith("fp64") else cu.MIXED, chebyshev=mode.startswith("chebyshev"))
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    err = np.abs(x - xd).max()
    assert err <= (1e-6 * np.abs(xd).max() if mode.endswith("fp64") else 1e-4), err
    _check_invariants(w, A, w.power, x, res)


@pytest.mark.parametrize("precond", ["jacobi", "chebyshev"])
def test_cfg5_full_size_200_steps(precond):
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(5)
    A = O.assemble_workload(w)
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.Solver(M, cu.Opts(precision=cu.MIXED, rtol=1e-8, true_resid_period=5))
    if precond == "chebyshev":      # setup once, reused by all 200 steps
        S.setup_chebyshev(to_dev(W.power_for_step(w, 1)), lanczos_steps=40, degree=30)
    T = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    cap = np.repeat(w.cvol * (w.dx * w.dy * w.dz) / w.dt, w.nx * w.ny)
    T_prev = np.zeros(w.n)
    To = np.zeros(w.n)
    total_its = 0
    for step in range(1, w.n_steps + 1):
        P = W.power_for_step(w, step)
        S.step(to_dev(P), T)
        check = step <= 2 or step % 25 == 0 or step == w.n_steps
        if not check:
            continue
        res = S.result()
        assert res.status == 0, (step, res)
        total_its += res.iterations
        Tg = T.cpu().numpy()
        # this step alone: rhs from the GPU's own T_n (kept from the previous checked step only when adjacent)
        if step <= 2:
            bo = O.transient_rhs(w, P, To)
            ro = O.pcg(A, bo, x0=To, rtol=1e-8)
            assert ro.status == 0
            assert np.abs(Tg - ro.x).max() <= 1e-4
            To = ro.x
        # property checks valid at any step: the per-step energy balance cannot be formed without T_n, so
        # re-run one more step from the current state and verify THAT step against the direct solve
        Pn = W.power_for_step(w, step + 1000)
        T2 = T.clone()
        S.step(to_dev(Pn), T2)
        r2 = S.result()
        assert r2.status == 0
        b2 = O.transient_rhs(w, Pn, Tg)
        xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, b2, w.cvol, w.dt)
        T2h = T2.cpu().numpy()
        assert np.abs(T2h - xd).max() <= 1e-4, step
        rel = np.linalg.norm(b2 - O.spmv(A, T2h)) / np.linalg.norm(b2)
        assert rel <= 1e-8
        top = T2h.reshape(w.nz, -1)[w.nz - 1]
        lhs = (cap * (T2h - Tg)).sum() + (w.h_top * w.dx * w.dy) * top.sum()
        assert lhs == pytest.approx(Pn.sum(), rel=1e-6)
    assert total_its > 0
    S.close()
