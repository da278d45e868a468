"""The operators the preconditioner multiplies by in the reduced-storage modes, as CSR matrices in fp64 --
TEST INFRASTRUCTURE, NOT PRODUCT CODE.

PAPER.md:219: "A2 ... single", "A3 ... half" copies of the Quad-Diag matrix; Alg. 4:
entries are LOADED in the narrow type and PROMOTED before the arithmetic ("arithmetic decoupling").  What the narrow
storage does to the operator is therefore exactly a rounding of each stored entry; everything after the promotion is
ordinary arithmetic.  These functions build that rounded operator explicitly, so that Alg. 3 evaluated on it in fp64
(oracle_cheb_apply) is an element-by-element reference for the fp32 kernels: what remains between the two is fp32
rounding of the vector arithmetic only.

Readings: the operator is applied in DIFFERENCE form (R-F3), i.e. the main diagonal is not a
stored entry but s_i + sum_j g_ij with the exact row sums s; the half-precision copy stores S * entry with S the power
of two that brings the largest |off-diagonal| into [2^13, 2^14) (fp16's normal range starts at 6e-5, the entries here
are 1e-8 ... 1e-3 W/K), and 1/S is applied after the promotion -- exact, S being a power of two.
Imports only numpy and the oracle's CSR container.
"""
from __future__ import annotations

import numpy as np

from . import oracle as O


def _rows(A: O.CSR) -> np.ndarray:
    return np.repeat(np.arange(A.n), np.diff(A.rowptr))


def _difference_form(A: O.CSR, row_sums, offdiag_rounded: np.ndarray) -> O.CSR:
    rows = _rows(A)
    offd = A.col != rows
    val = A.val.copy()
    val[offd] = offdiag_rounded
    neg = np.zeros(A.n)
    np.add.at(neg, rows[offd], val[offd])
    val[~offd] = np.asarray(row_sums, dtype=np.float64) - neg          # s_i + sum_j g_ij, g = -offdiag
    return O.CSR(A.n, A.rowptr, A.col, val)


def fp32_difference_operator(A: O.CSR, row_sums) -> O.CSR:
    """A2 in difference form: off-diagonals rounded to fp32 (round-to-nearest-even)."""
    offd = A.col != _rows(A)
    return _difference_form(A, row_sums, A.val[offd].astype(np.float32).astype(np.float64))


def fp16_scale(A: O.CSR) -> float:
    """The power of two S with S * max|off-diagonal| in [2^13, 2^14)."""
    offd = A.col != _rows(A)
    m = float(np.abs(A.val[offd]).max())
    _, e = np.frexp(m)                       # m = f * 2^e, f in [0.5, 1)
    return float(np.ldexp(1.0, 14 - int(e)))


def fp16_difference_operator(A: O.CSR, row_sums) -> O.CSR:
    """A3 (Alg. 4 lines 6-8) in difference form: off-diagonals stored as fp16(S * entry),
    promoted and multiplied by 1/S."""
    offd = A.col != _rows(A)
    S = fp16_scale(A)
    return _difference_form(A, row_sums, (A.val[offd] * S).astype(np.float16).astype(np.float64) / S)
