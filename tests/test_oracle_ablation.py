"""Pins of oracle/ablation.py (CPU).  In fp64 the fixed-precision loop IS Alg. 1 and must reproduce oracle_pcg (the C++
oracle, itself pinned by direct solves); in fp32 it must show what the paper's Table VI shows for fixed FP32
(the loop "converges" at about the fp64 iteration count while the answer has drifted) and what SURVEY
F2 measured on these grids (true residual floor ~1e-2 ||b||, temperature error >= 1e-2 K)."""
import numpy as np

import workloads as W
from oracle import oracle as O
from oracle import ablation as AB
from direct_solve import solve_layered


def test_fp64_instance_reproduces_oracle_pcg():
    for kw in (dict(cfg=1), dict(cfg=6, nx=20, ny=18, nz=10, n_hot=3)):
        w = W.make_workload(**kw)
        A = O.assemble_workload(w)
        ref = O.pcg(A, w.power, rtol=1e-8)
        res = AB.pcg_fixed(A, w.power, dtype=np.float64, rtol=1e-8)
        assert res.status == 7 and abs(res.iterations - ref.iterations) <= 1
        assert np.abs(res.x - ref.x).max() <= 1e-7 * np.abs(ref.x).max()
        assert res.rel_resid_true <= 1.5e-8                       # unverified, but in fp64 the two residuals agree
        un = AB.pcg_fixed(A, w.power, dtype=np.float64, rtol=1e-8, precond=0)
        assert np.abs(un.x - ref.x).max() <= 1e-6 * np.abs(ref.x).max()


def test_fixed_fp32_drifts_like_table_vi():
    w = W.make_workload(2, nx=64, ny=64, nz=16, n_hot=8)
    A = O.assemble_workload(w)
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    ref = O.pcg(A, w.power, rtol=1e-8)
    res = AB.pcg_fixed(A, w.power, dtype=np.float32, rtol=1e-6, max_iters=5000)
    err = np.abs(res.x - xd).max()
    # the loop is satisfied (or stalls at the fp32 floor of its own residual) ...
    assert res.status in (7, 1) and res.rel_resid_rec <= 1e-4
    # ... while the answer is wrong by far more than the 1e-4 K bar and the true residual sits at a floor
    assert err >= 1e-2, err
    assert res.rel_resid_true >= 1e-4
    assert res.rel_resid_true >= 100 * res.rel_resid_rec
    assert np.abs(ref.x - xd).max() <= 1e-6 * np.abs(xd).max()    # fp64 on the same system is fine
    assert AB.pcg_fixed(A, np.zeros(w.n)).iterations == 0


def test_lanczos_fixed_fp64_reproduces_oracle_lanczos_and_fp32_stays_close():
    """Lanczos in FP32 on the fixed-FP32 SpMV.  The fp64 instance of the step-by-step reference is the C++
    oracle's recurrence (same alpha, beta); the fp32 instance gives the same spectral interval to a per cent or two --
    which is all the preconditioner needs."""
    for kw in (dict(cfg=1), dict(cfg=3, nx=20, ny=16, nz=16, n_hot=4)):
        w = W.make_workload(**kw)
        A = O.assemble_workload(w)
        a64, b64 = O.lanczos(A, w.power, 25)
        a, b = AB.lanczos_fixed(A, w.power, 25, dtype=np.float64)
        assert np.allclose(a, a64, rtol=1e-8, atol=0) and np.allclose(b[:-1], b64[:-1], rtol=1e-7, atol=0)
        a32, b32 = AB.lanczos_fixed(A, w.power, 25, dtype=np.float32)
        lo, hi = O.ritz_extremes(a64, b64)
        lo32, hi32 = O.ritz_extremes(a32, b32)
        assert abs(hi32 - hi) <= 0.02 * hi          # unconverged Ritz values after 25 steps move with the rounding
        assert abs(lo32 - lo) <= 0.05 * lo
        assert np.abs(a32[:5] - a64[:5]).max() <= 1e-5 * np.abs(a64).max()      # the first steps agree to fp32 rounding
