"""Pins of the step-by-step mixed-precision reference (oracle/policy.py), CPU only.

What fixes it independently of itself: the converged x must be A^-1 b (dense Cholesky / direct solve), the
true residual must meet rtol, the early-stage operator must keep the exact row sums (closed form A~ 1 = s) and
be an fp32-sized perturbation of A, and with an operator that needs no promotion-by-drift the switch must be
the (14a) one at the first iteration whose recursive residual is below sqrt(rtol) ||b||."""
import numpy as np
import pytest
import scipy.linalg as sla

import workloads as W
from oracle import oracle as O
from oracle import policy as P
from direct_solve import solve_layered


def row_sums(w):
    s = np.zeros((w.nz, w.nx * w.ny))
    s[w.nz - 1] += w.h_top * w.dx * w.dy
    if w.transient:
        s += (w.cvol * (w.dx * w.dy * w.dz) / w.dt)[:, None]
    return s.reshape(-1)


def test_early_operator_keeps_row_sums_and_is_fp32_close():
    w = W.make_workload(3, nx=14, ny=11, nz=16, n_hot=4)
    A = O.assemble_workload(w)
    s = row_sums(w)
    A2 = P.early_stage_operator(A, s)
    ones = O.spmv(A2, np.ones(w.n))
    assert np.abs(ones - s).max() <= 1e-12 * np.abs(A.val).max()          # A~ 1 = s (difference form)
    M, M2 = A.to_scipy().toarray(), A2.to_scipy().toarray()
    off = ~np.eye(w.n, dtype=bool)
    assert np.abs(M2[off] - M[off]).max() <= 2 ** -24 * np.abs(M[off]).max() * 1.01
    assert np.array_equal(M2, M2.T)


@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=2, nx=40, ny=36, nz=16, n_hot=6)])
def test_mixed_reference_converges_to_the_direct_solution(kw):
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, period=20)
    assert res.status == 0 and res.rel_resid_true <= 1e-8
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    assert np.abs(res.x - xd).max() <= 1e-4
    assert np.linalg.norm(w.power - O.spmv(A, res.x)) <= 1e-8 * np.linalg.norm(w.power)
    assert res.promotions == 1 and res.switch_reason == 1                 # (14a) fires first on these grids
    ref = O.pcg(A, w.power, rtol=1e-8, hist_len=5000)
    first = int(np.argmax(ref.hist[:ref.iterations + 1] <= 1e-4))         # first iteration with ||r|| <= sqrt(rtol) ||b||
    assert abs(res.switch_iteration - first) <= 2
    assert abs(res.iterations - ref.iterations) <= max(3, 0.03 * ref.iterations)   # soft restart: no penalty


def test_mixed_reference_tiny_vs_cholesky_and_zero_rhs():
    w = W.make_workload(1, nx=6, ny=5, nz=4, n_hot=1)
    A = O.assemble_workload(w)
    xs = sla.cho_solve(sla.cho_factor(A.to_scipy().toarray()), w.power)
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-9, period=5)
    assert res.status == 0 and np.abs(res.x - xs).max() <= 1e-6 * np.abs(xs).max()
    z = P.pcg_mixed(A, row_sums(w), np.zeros(w.n), x0=np.ones(w.n))
    assert z.status == 0 and z.iterations == 0 and np.all(z.x == 0)
