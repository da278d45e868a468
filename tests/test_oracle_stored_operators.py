"""Pins of oracle/stored_operators.py (CPU): the rounded operators are what PAPER.md:219 / Alg. 4 say they are --
each off-diagonal within half an ulp of the narrow type of the exact one, symmetric, exact row sums (difference form,
R-F3), SPD -- and the fp16 scale is the stated power of two."""
import numpy as np

import workloads as W
from oracle import oracle as O
from oracle import stored_operators as SO


def _row_sums(w):
    s = np.zeros((w.nz, w.nx * w.ny))
    s[w.nz - 1] += w.h_top * w.dx * w.dy
    if w.transient:
        s += (w.cvol * (w.dx * w.dy * w.dz) / w.dt)[:, None]
    return s.reshape(-1)


def test_rounded_operators_are_half_ulp_copies_with_exact_row_sums():
    for kw in (dict(cfg=3, nx=10, ny=7, nz=6, n_hot=2), dict(cfg=6, nx=9, ny=8, nz=10, n_hot=2),
               dict(cfg=5, nx=8, ny=6, nz=4, n_hot=1)):
        w = W.make_workload(**kw)
        A = O.assemble_workload(w)
        s = _row_sums(w)
        M = A.to_scipy().toarray()
        off = ~np.eye(w.n, dtype=bool)
        nz = off & (M != 0)
        for op, ulp_half in ((SO.fp32_difference_operator(A, s), 2.0 ** -24), (SO.fp16_difference_operator(A, s), 2.0 ** -11)):
            R = op.to_scipy().toarray()
            assert np.array_equal(R, R.T)
            assert np.array_equal(R != 0, M != 0)                              # no entry flushed to zero, none created
            assert (np.abs(R[nz] - M[nz]) <= ulp_half * np.abs(M[nz]) * (1 + 1e-12)).all()
            assert np.abs(R @ np.ones(w.n) - s).max() <= 1e-12 * np.abs(M).max()   # A~ 1 = s
            assert np.linalg.eigvalsh(R).min() > 0
        S = SO.fp16_scale(A)
        m = np.abs(M[off]).max()
        assert np.log2(S) == int(np.log2(S)) and 2.0 ** 13 <= S * m < 2.0 ** 14
        # fp16 really is the storage type: every stored value S * entry is an fp16 number
        R16 = SO.fp16_difference_operator(A, s).to_scipy().toarray()
        st = R16[nz] * S
        assert np.array_equal(st.astype(np.float16).astype(np.float64), st)
        # and it differs from the fp32 copy (2^-11 vs 2^-24)
        assert np.abs(R16[nz] - M[nz]).max() > 10 * np.abs(SO.fp32_difference_operator(A, s).to_scipy().toarray()[nz] - M[nz]).max()


def test_fp32_difference_operator_is_the_policy_early_operator():
    from oracle import policy as P
    w = W.make_workload(3, nx=10, ny=7, nz=6, n_hot=2)
    A = O.assemble_workload(w)
    s = _row_sums(w)
    assert np.array_equal(SO.fp32_difference_operator(A, s).val, P.early_stage_operator(A, s).val)
