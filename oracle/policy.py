"""Step-by-step CPU reference of the adaptive mixed-precision PCG -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Follows PAPER.md §IV-D in the paper's order, with the readings of DESIGN.md §3:
  * early stage: Alg. 1 with the SpMV of line 6 on the fp32-STORED matrix promoted to
    fp64 ("FP64/32 SpMV with AD") in difference form (R-F3); x, r, p, dots in fp64;
  * every T iterations r_true = b - A1 x in fp64, then the switch criteria in this order:
    recursive residual converged, (14a) relative (R-G8), (14c) second print (R-G10), (14b) on successive
    evaluations and only when the recursive residual did decrease (R-G9);
  * hot restart (R-G11): r := r_true; p from its defining equation -- Alg. 1 line 12 with
    beta = rho(new r)/rho_k while the drift is small, Alg. 1 line 3 (p = z) when it is large;
  * late stage: fp64 operator; exit only on a verified true residual (R-G7).
Plain numpy + the oracle's CSR SpMV; no blocking, no fusion.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import oracle as O


@dataclass
class MixedResult:
    x: np.ndarray
    status: int            # 0 converged, 1 max_iters, 2 breakdown
    iterations: int
    promotions: int
    true_resid_evals: int
    switch_reason: int     # 0 none, 1 (14a), 2 (14b), 3 (14c), 4 recursive converged
    switch_iteration: int
    rel_resid_true: float


def early_stage_operator(A: O.CSR, row_sums: np.ndarray) -> O.CSR:
    """The matrix the early stage multiplies by: off-diagonals rounded to fp32 (A2), diagonal
    rebuilt so that every row keeps its exact row sum s_i (difference form, R-F3)."""
    val = A.val.copy()
    n = A.n
    rows = np.repeat(np.arange(n), np.diff(A.rowptr))
    offd = A.col != rows
    val[offd] = val[offd].astype(np.float32).astype(np.float64)
    neg_sum = np.zeros(n)
    np.add.at(neg_sum, rows[offd], val[offd])
    val[~offd] = row_sums - neg_sum            # s_i + sum_j g_ij, g = -offdiag
    return O.CSR(n, A.rowptr, A.col, val)


def pcg_mixed(A: O.CSR, row_sums, b, x0=None, rtol=1e-8, period=20, max_iters=200000,
              soft_drift=0.1) -> MixedResult:
    n = A.n
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(n) if x0 is None else np.array(x0, dtype=np.float64)
    dg = np.empty(n)
    rows = np.repeat(np.arange(n), np.diff(A.rowptr))
    dg[:] = A.val[A.col == rows]
    A2 = early_stage_operator(A, np.asarray(row_sums, dtype=np.float64))
    bb = float(b @ b)
    if bb == 0.0:
        return MixedResult(np.zeros(n), 0, 0, 0, 0, 0, 0, 0.0)
    tol2, sw2 = rtol * rtol * bb, rtol * bb
    r = b - O.spmv(A, x)                                   # Alg. 1 line 1
    rr = float(r @ r)
    tt = rr
    if rr <= tol2:
        return MixedResult(x, 0, 0, 0, 0, 0, 0, np.sqrt(rr / bb))
    z = r / dg                                             # line 2 (Jacobi, R-G6)
    p = z.copy()                                           # line 3
    rho = float(r @ z)
    early, it, since, promotions, evals = True, 0, 0, 0, 0
    reason_sw, it_sw = 0, 0
    tt_prev, rr_prev_eval = rr, rr
    status = 1
    while True:
        mu = O.spmv(A2 if early else A, p)                 # line 6
        pmu = float(p @ mu)
        if not (pmu > 0.0) or not np.isfinite(pmu):
            status = 2
            break
        alpha = rho / pmu                                  # line 7
        x += alpha * p                                     # line 8
        r -= alpha * mu                                    # line 9
        z = r / dg                                         # line 10
        rho_new = float(r @ z)
        beta = rho_new / rho                               # line 11
        rho = rho_new
        rr = float(r @ r)
        it += 1                                            # line 13
        since += 1
        conv_rec = rr <= tol2
        want = conv_rec or (early and rr <= sw2) or (early and since >= period) or it >= max_iters
        restart = 0
        if want:
            t = b - O.spmv(A, x)                           # r_true
            tt = float(t @ t)
            dd = float((t - r) @ (t - r))
            evals += 1
            since = 0
            if tt <= tol2:
                status = 0
                break
            if it >= max_iters:
                status = 1
                break
            if not early:
                if conv_rec:
                    restart = 1
            else:
                reason = 0
                if conv_rec:
                    reason = 4
                elif rr <= sw2:
                    reason = 1                             # (14a)
                elif dd >= 0.25 * tt:
                    reason = 3                             # (14c)
                elif tt > 0.81 * tt_prev and rr <= 0.81 * rr_prev_eval:
                    reason = 2                             # (14b)
                if reason:
                    early = False
                    promotions += 1
                    reason_sw, it_sw = reason, it
                    restart = 2 if dd <= soft_drift * soft_drift * tt else 1
            tt_prev, rr_prev_eval = tt, rr
            if restart:                                    # hot restart
                r = t
                z = r / dg
                rho_t = float(r @ z)
                beta = beta * (rho_t / rho) if (restart == 2 and rho > 0.0) else 0.0
                rho = rho_t
                rr = tt
        p = z + beta * p                                   # line 12 (line 3 when beta = 0)
    return MixedResult(x, status, it, promotions, evals, reason_sw, it_sw, float(np.sqrt(tt / bb)))
