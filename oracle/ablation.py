"""Fixed-precision PCG, step by step -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

PAPER.md:336 ("Fixed-Precision SpMV: Standard FP64 and FP32 kernels implemented directly via Algorithm 2") and the
fixed-FP32 column of Table VI: Alg. 1 with EVERY object in one working precision
-- the matrix (A2 = the stored entries rounded to that precision, standard form), x, r, z, p, mu, alpha, beta and the
three inner products -- M = diag(A2).  The loop stops on its own recursive residual, ||r||_2 <= rtol ||b||_2 (Alg. 1
line 5, relative form R-G7), and never evaluates b - A x: that is the paper's point ("numerical drift").
`dtype=np.float64` is the same code in double precision and must reproduce oracle_pcg; that pins the loop.
Plain numpy; the SpMV is scipy's CSR product in the working precision (a library primitive).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import oracle as O


@dataclass
class FixedResult:
    x: np.ndarray            # widened to fp64
    status: int              # 7 = recursive residual passed (unverified), 1 = max_iters, 2 = breakdown, 0 = b == 0
    iterations: int
    rel_resid_rec: float     # what the loop believes
    rel_resid_true: float    # ||b - A1 x||_2 / ||b||_2 evaluated in fp64 afterwards, for the report only


def pcg_fixed(A: O.CSR, b, dtype=np.float32, rtol=1e-8, max_iters=200000, precond=1, x0=None) -> FixedResult:
    T = np.dtype(dtype).type
    n = A.n
    S = A.to_scipy().astype(dtype)                       # A2: every stored entry rounded to the working precision
    dg = S.diagonal()
    b64 = np.asarray(b, dtype=np.float64)
    bw = b64.astype(dtype)
    x = np.zeros(n, dtype=dtype) if x0 is None else np.asarray(x0, dtype=np.float64).astype(dtype)
    bb = T(bw @ bw)
    if bb == 0:
        return FixedResult(np.zeros(n), 0, 0, 0.0, 0.0)
    r = bw - S @ x                                       # line 1
    z = r / dg if precond else r.copy()                  # line 2
    p = z.copy()                                         # line 3
    rho = T(r @ z)
    rr = T(r @ r)
    tol2 = T(rtol) * T(rtol) * bb
    it, status = 0, 1
    if rr <= tol2:
        status = 7
    while status == 1 and it < max_iters:                # line 5
        mu = S @ p                                       # line 6
        pmu = T(p @ mu)
        if not (pmu > 0) or not np.isfinite(pmu):
            status = 2
            break
        alpha = T(rho / pmu)                             # line 7
        x = x + alpha * p                                # line 8
        r = r - alpha * mu                               # line 9
        z = r / dg if precond else r                     # line 10
        rho_new = T(r @ z)
        beta = T(rho_new / rho)                          # line 11
        rho = rho_new
        rr = T(r @ r)
        it += 1                                          # line 13
        if not np.isfinite(rr):
            status = 2
            break
        if rr <= tol2:
            status = 7
            break
        p = z + beta * p                                 # line 12
    x64 = x.astype(np.float64)
    t = b64 - O.spmv(A, x64)
    return FixedResult(x64, status, it, float(np.sqrt(float(rr) / float(bb))),
                       float(np.linalg.norm(t) / np.linalg.norm(b64)))


def lanczos_fixed(A: O.CSR, v0, m: int, dtype=np.float32):
    """m Lanczos steps entirely in one working precision on A2 = the stored entries rounded to that
    precision, standard form ("the N-step Lanczos algorithm ... in FP32 precision using the fixed FP32 SpMV
    kernel").  Same recurrence as oracle_lanczos (C++): v normalised, no reorthogonalisation; returns alpha[m'], beta[m'].
    `dtype=np.float64` must reproduce oracle_lanczos; that pins the recurrence."""
    T = np.dtype(dtype).type
    S = A.to_scipy().astype(dtype)
    v = np.asarray(v0, dtype=np.float64).astype(dtype)
    v = v / T(np.sqrt(T(v @ v)))
    vp = np.zeros_like(v)
    bprev = T(0)
    alpha, beta = [], []
    for _ in range(m):
        w = S @ v - bprev * vp
        a = T(w @ v)
        w = w - a * v
        b = T(np.sqrt(T(w @ w)))
        alpha.append(float(a))
        beta.append(float(b))
        if not b > 0:
            break
        vp, v = v, w / b
        bprev = b
    return np.array(alpha), np.array(beta)
