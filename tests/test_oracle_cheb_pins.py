"""Pins of the oracle's Chebyshev preconditioner, Lanczos and PCG-Chebyshev.

Alg. 3 is pinned to the closed form the paper derives it from: after k steps the
residual polynomial is P_k(lambda) = C_k((theta - lambda)/delta) / C_k(theta/delta) (eq. (11a),
PAPER.md:263), C_k from the three-term recurrence eq. (12), evaluated here on the
eigen-decomposition of a tiny matrix (eq. (8)) -- none of which the oracle uses.
"""
import numpy as np
import pytest
import scipy.linalg as sla

import workloads as W
from oracle import oracle as O
from test_oracle_pins import _rand_problem


def _cheb_C(k, t):
    c0, c1 = np.ones_like(t), t.copy()                      # eq. (12)
    if k == 0:
        return c0
    for _ in range(k - 1):
        c0, c1 = c1, 2 * t * c1 - c0
    return c1


@pytest.mark.parametrize("k", [1, 2, 5, 30])
def test_cheb_apply_equals_closed_form_polynomial(k):
    A, b, _ = _rand_problem(5, 4, 3, 21)
    M = A.to_scipy().toarray()
    lam, V = np.linalg.eigh(M)
    lmin, lmax = lam[0] * 0.9, lam[-1] * 1.05
    theta, delta = (lmax + lmin) / 2, (lmax - lmin) / 2
    Pk = _cheb_C(k, (theta - lam) / delta) / _cheb_C(k, np.array([theta / delta]))[0]   # eq. (11a)
    q = (1.0 - Pk) / lam                                    # z = A^-1 (r - P_k(A) r)
    z_ref = V @ (q * (V.T @ b))
    z = O.cheb_apply(A, b, lmin, lmax, k)
    assert np.abs(z - z_ref).max() <= 1e-9 * np.abs(z_ref).max()
    # minimax property eq. (9)-(10): |P_k| <= 1/C_k(theta/delta) on [lmin, lmax]
    assert np.abs(Pk).max() <= 1.0 / _cheb_C(k, np.array([theta / delta]))[0] * (1 + 1e-9)


def test_cheb_apply_is_linear_symmetric_positive():
    A, b, _ = _rand_problem(4, 3, 2, 22)
    n = A.n
    M = A.to_scipy().toarray()
    lam = np.linalg.eigvalsh(M)
    Q = np.column_stack([O.cheb_apply(A, e, lam[0], lam[-1] * 1.05, 7) for e in np.eye(n)])
    assert np.abs(Q - Q.T).max() <= 1e-9 * np.abs(Q).max()          # q(A) is symmetric
    assert np.linalg.eigvalsh((Q + Q.T) / 2).min() > 0              # and positive definite
    x = W.normal01(22, 20, 21, np.arange(n))
    assert np.allclose(O.cheb_apply(A, x, lam[0], lam[-1] * 1.05, 7), Q @ x, rtol=1e-9, atol=0)


def test_lanczos_ritz_values_vs_dense_eigenvalues():
    A, b, _ = _rand_problem(5, 4, 3, 23)
    M = A.to_scipy().toarray()
    lam = np.linalg.eigvalsh(M)
    a, bt = O.lanczos(A, b, 25)
    lo, hi = O.ritz_extremes(a, bt)
    assert lam[0] * (1 - 1e-9) <= lo and hi <= lam[-1] * (1 + 1e-9)   # Ritz values lie inside the spectrum
    assert hi >= 0.99 * lam[-1]                                     # and the top converges quickly
    # T = V^T A V: alpha_0 = v0^T A v0 / v0^T v0
    assert a[0] == pytest.approx(b @ (M @ b) / (b @ b), rel=1e-12)


@pytest.mark.parametrize("dims", [(5, 4, 3), (9, 8, 6)])
def test_pcg_cheb_vs_dense_cholesky(dims):
    A, b, _ = _rand_problem(*dims, 24)
    M = A.to_scipy().toarray()
    xs = sla.cho_solve(sla.cho_factor(M), b)
    lam = np.linalg.eigvalsh(M)
    # interval [lambda_max/400, 1.02 lambda_max]: the upper end must bound the spectrum (q(A) SPD); the lower
    # end need not reach lambda_min (DESIGN.md R-C2)
    # rtol 1e-10 and the 1e-8 bar are the ones this pin was written with (round 1 had loosened them to 1e-9 / 1e-7 together
    # with the change of interval, which only the interval needed: VERDICT r1); measured error 4e-12 / 3e-13
    r = O.pcg_cheb(A, b, lam[-1] / 400, 1.02 * lam[-1], 8, rtol=1e-10, max_iters=2000)
    assert r.status == 0 and r.rel_resid_true <= 1e-10
    assert np.abs(r.x - xs).max() <= 1e-8 * np.abs(xs).max()
    r0 = O.pcg(A, b, rtol=1e-9, max_iters=5000, precond=0)
    assert r.iterations < r0.iterations                            # fewer outer iterations than plain CG


def test_pcg_cheb_cfg1_iterations_and_solution():
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    a, bt = O.lanczos(A, w.power, 40)
    lo, hi = O.ritz_extremes(a, bt)
    r = O.pcg_cheb(A, w.power, lo, 1.05 * hi, 30)
    rj = O.pcg(A, w.power)
    assert r.status == 0 and r.rel_resid_true <= 1e-8
    assert r.iterations < rj.iterations / 4                        # Table VII: 44-107 vs 647-1593
    assert np.abs(r.x - rj.x).max() <= 1e-6 * np.abs(rj.x).max()
