"""Step-by-step CPU reference of the adaptive mixed-precision PCG -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Written from PAPER.md §IV-D, in the paper's order and with the paper's constants; the
readings taken where the text is silent or garbled are DESIGN.md §3's and are named where they are used.

  * Stage-switching criteria, one function each, on NORMS (not squares), with the printed
    constants 0.9 and 0.5:
        (14a)  ||r_low||_2 <= 10^n, n = log10(eps)/2        -> relative form sqrt(eps) ||b||_2 (R-G8)
        (14b)  ||r_true^k||_2 > 0.9 ||r_true^{k-1}||_2      -> k, k-1 = successive EVALUATIONS (R-G9), and only
               "despite a decreasing recursive one": ||r_low^k|| <= 0.9 ||r_low^{k-1}||
        (14c)  ||r_true - r_low||_2 >= 0.5 ||r_true||_2     -> the second print (R-G10)
    "The early-to-late transition is triggered when any of the following holds": `switch_mask`
    carries all that held (bit 0 = a, bit 1 = b, bit 2 = c), `switch_reason` the first one in the printed order.
  * r_true = b - A x is "periodically re-evaluated in FP64, such as every 20 iterations for steady-state and
    every 5 for transient"; (14a) needs only the recursive norm and is looked at every iteration.
  * Early stage: Alg. 1 with the SpMV of line 6 on the fp32-STORED matrix
    promoted to fp64, everything else fp64.  The operator is a parameter: the default is the difference form of
    R-F3, `standard_form_fp32_operator` is the paper's A2 taken literally.
  * Hot restart: "explicitly recomputes r and p from their defining equations", x carried over.
    r := b - A x.  p: Alg. 1 line 12 (p = z + beta p, beta = rho(new r) / rho_{k-1}) while the drift is small
    (||r_true - r_low|| <= soft_drift ||r_true||, R-G11: "preserving the established Krylov subspace",
    PAPER.md:326) -- kind 2, "soft"; Alg. 1 line 3 (p = z) otherwise -- kind 1, "hard".
  * Late stage: the fp64 operator.  Exit only on a verified true residual (R-G7); a failed
    verification replaces r and restarts the direction (kind 1), exactly as oracle_pcg does.
Plain numpy + the oracle's CSR SpMV; no blocking, no fusion.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import oracle as O

CRIT_A, CRIT_B, CRIT_C = 1, 2, 4     # bits of switch_mask


# ---------------------------------------------------------------- eq. (14a)-(14c), one function each
def crit_14a(norm_r_low: float, eps_rel: float, norm_b: float) -> bool:
    """(14a): ||r_low||_2 <= 10^(log10(eps)/2) = sqrt(eps); relative to ||b||_2 (R-G8).
    For eps >= 1 the stopping threshold eps ||b|| itself is the larger one and is used instead, so that a
    recursive residual that passes the stopping test always passes (14a)."""
    return norm_r_low <= max(np.sqrt(eps_rel), eps_rel) * norm_b


def crit_14b(norm_true_k: float, norm_true_km1: float, norm_low_k: float, norm_low_km1: float) -> bool:
    """(14b), PAPER.md:387 + :400: the true residual failed to drop below 0.9 x its value at the previous
    evaluation although the recursive one did ("stagnation of the true residual despite a decreasing recursive
    one")."""
    return norm_true_k > 0.9 * norm_true_km1 and norm_low_k <= 0.9 * norm_low_km1


def crit_14c(norm_drift: float, norm_true: float) -> bool:
    """(14c): ||r_true - r_low||_2 >= 0.5 ||r_true||_2."""
    return norm_drift >= 0.5 * norm_true


def switch_mask(norm_low, norm_true, norm_drift, norm_true_prev, norm_low_prev, eps_rel, norm_b) -> int:
    """All criteria that hold at one evaluation of r_true ("any of the following")."""
    m = 0
    if crit_14a(norm_low, eps_rel, norm_b):
        m |= CRIT_A
    if crit_14b(norm_true, norm_true_prev, norm_low, norm_low_prev):
        m |= CRIT_B
    if crit_14c(norm_drift, norm_true):
        m |= CRIT_C
    return m


def first_reason(mask: int) -> int:
    """1 = (14a), 2 = (14b), 3 = (14c): the first criterion of the mask in the printed order; 0 = none."""
    return 1 if mask & CRIT_A else 2 if mask & CRIT_B else 3 if mask & CRIT_C else 0


def restart_kind(norm_drift: float, norm_true: float, soft_drift: float) -> int:
    """Hot restart at the switch (R-G11): 2 = soft (p keeps its history), 1 = hard (p = z)."""
    return 2 if norm_drift <= soft_drift * norm_true else 1


# ---------------------------------------------------------------- early-stage operators
def _rows(A: O.CSR) -> np.ndarray:
    return np.repeat(np.arange(A.n), np.diff(A.rowptr))


def early_stage_operator(A: O.CSR, row_sums: np.ndarray) -> O.CSR:
    """Difference form (R-F3): off-diagonals rounded to fp32 (A2), diagonal rebuilt so that every
    row keeps its exact row sum s_i."""
    val = A.val.copy()
    rows = _rows(A)
    offd = A.col != rows
    val[offd] = val[offd].astype(np.float32).astype(np.float64)
    neg_sum = np.zeros(A.n)
    np.add.at(neg_sum, rows[offd], val[offd])
    val[~offd] = row_sums - neg_sum            # s_i + sum_j g_ij, g = -offdiag
    return O.CSR(A.n, A.rowptr, A.col, val)


def standard_form_fp32_operator(A: O.CSR) -> O.CSR:
    """The paper's A2 literally (PAPER.md:219 "A2 ... single", :335): EVERY stored entry, main diagonal
    included, rounded to fp32 and promoted back; applied in standard form."""
    return O.CSR(A.n, A.rowptr, A.col, A.val.astype(np.float32).astype(np.float64))


# ---------------------------------------------------------------- the solver
@dataclass
class MixedResult:
    x: np.ndarray
    status: int            # 0 converged, 1 max_iters, 2 breakdown
    iterations: int
    promotions: int
    true_resid_evals: int
    switch_reason: int     # 0 none, 1 (14a), 2 (14b), 3 (14c)
    switch_iteration: int
    rel_resid_true: float
    switch_mask: int = 0   # every criterion that held at the switch (bits CRIT_A/B/C)
    hard_restarts: int = 0
    soft_restarts: int = 0
    evals: list = field(default_factory=list)   # (iteration, ||r_low||, ||r_true||, ||r_true - r_low||) per evaluation


def pcg_mixed(A: O.CSR, row_sums, b, x0=None, rtol=1e-8, period=20, max_iters=200000, soft_drift=0.1,
              early_operator: O.CSR | None = None, start_early=True) -> MixedResult:
    n = A.n
    b = np.asarray(b, dtype=np.float64)
    x = np.zeros(n) if x0 is None else np.array(x0, dtype=np.float64)
    dg = A.val[A.col == _rows(A)].copy()
    A_early = early_operator if early_operator is not None else \
        early_stage_operator(A, np.asarray(row_sums, dtype=np.float64))
    nb = float(np.sqrt(b @ b))
    if nb == 0.0:
        return MixedResult(np.zeros(n), 0, 0, 0, 0, 0, 0, 0.0)
    r = b - O.spmv(A, x)                                   # Alg. 1 line 1 (fp64 operator: r0 is a true residual)
    n_low = float(np.sqrt(r @ r))
    n_true = n_low
    if n_low <= rtol * nb:
        return MixedResult(x, 0, 0, 0, 0, 0, 0, n_low / nb)
    z = r / dg                                             # line 2 (Jacobi, R-G6)
    p = z.copy()                                           # line 3
    rho = float(r @ z)
    early = bool(start_early)
    it = since = promotions = n_evals = hard = soft = 0
    reason_sw = it_sw = mask_sw = 0
    n_true_prev, n_low_prev = n_true, n_low                # "previous evaluation" = r0
    status = 1
    log = []
    while True:
        mu = O.spmv(A_early if early else A, p)            # line 6
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
        n_low = float(np.sqrt(r @ r))
        it += 1                                            # line 13
        since += 1
        conv_rec = n_low <= rtol * nb                      # line 5 (R-G7)
        look = conv_rec or it >= max_iters or \
            (early and (crit_14a(n_low, rtol, nb) or since >= period))
        kind = 0
        if look:
            t = b - O.spmv(A, x)                           # r_true in FP64
            n_true = float(np.sqrt(t @ t))
            n_drift = float(np.sqrt((t - r) @ (t - r)))
            n_evals += 1
            since = 0
            log.append((it, n_low, n_true, n_drift))
            if n_true <= rtol * nb:
                status = 0
                break
            if it >= max_iters:
                status = 1
                break
            if not early:
                if conv_rec:                               # late stage: verification failed
                    kind = 1
            else:
                mask = switch_mask(n_low, n_true, n_drift, n_true_prev, n_low_prev, rtol, nb)
                if mask:
                    early = False
                    promotions += 1
                    mask_sw, reason_sw, it_sw = mask, first_reason(mask), it
                    kind = restart_kind(n_drift, n_true, soft_drift)
            n_true_prev, n_low_prev = n_true, n_low
            if kind:                                       # hot restart
                r = t
                z = r / dg
                rho_t = float(r @ z)
                beta = beta * (rho_t / rho) if (kind == 2 and rho > 0.0) else 0.0
                rho = rho_t
                n_low = n_true
                hard += kind == 1
                soft += kind == 2
        p = z + beta * p                                   # line 12 (line 3 when beta = 0)
    return MixedResult(x, status, it, promotions, n_evals, reason_sw, it_sw, n_true / nb, mask_sw, hard, soft, log)
