"""Where must the stage switch of PAPER.md §IV-D happen?  Derived WITHOUT running any policy code: a textbook
PCG loop (Alg. 1, M = diag A) on the early-stage operator records x_k and the recursive residual
r_k; afterwards the history is scanned at the evaluation points k = T, 2T, ... and at every k for
(14a), with eq. (14a)-(14c) typed here from the paper, on norms.  Used by the CPU pins of
oracle/policy.py and by the GPU tests; imports only the oracle's CSR SpMV."""
import numpy as np

from oracle import oracle as O


def pcg_history(A_true, A_early, b, iters):
    """x_k, r_k (recursive) for k = 0..iters of Alg. 1 run entirely on A_early (x0 = 0, so r0 = b exactly)."""
    rows = np.repeat(np.arange(A_true.n), np.diff(A_true.rowptr))
    dg = A_true.val[A_true.col == rows]
    x = np.zeros(A_true.n)
    r = b.copy()
    z = r / dg
    p = z.copy()
    rho = r @ z
    xs, rs = [x.copy()], [r.copy()]
    for _ in range(iters):
        mu = O.spmv(A_early, p)
        alpha = rho / (p @ mu)
        x = x + alpha * p
        r = r - alpha * mu
        z = r / dg
        rho_new = r @ z
        p = z + (rho_new / rho) * p
        rho = rho_new
        xs.append(x.copy())
        rs.append(r.copy())
    return xs, rs


def expected_switch(A_true, A_early, b, rtol, T, iters):
    """(iteration, mask, margin): first evaluation at which any of (14a)-(14c) holds; mask bit 0/1/2 = a/b/c;
    margin = the smallest relative change of any compared quantity that would alter that outcome (no criterion
    firing earlier, the same set firing at the switch)."""
    xs, rs = pcg_history(A_true, A_early, b, iters)
    nb = np.linalg.norm(b)
    t_prev = l_prev = nb                                   # previous evaluation = r0 = b
    margin = np.inf
    since = 0
    for k in range(1, iters + 1):
        since += 1
        low = np.linalg.norm(rs[k])
        a = low <= np.sqrt(rtol) * nb                      # (14a), every iteration
        margin_a = abs(low / (np.sqrt(rtol) * nb) - 1.0)
        if not a and since < T:
            margin = min(margin, margin_a)
            continue
        since = 0
        t = b - O.spmv(A_true, xs[k])
        true = np.linalg.norm(t)
        drift = np.linalg.norm(t - rs[k])
        qt, ql, qc = true / (0.9 * t_prev), low / (0.9 * l_prev), drift / (0.5 * true)
        bcrit = qt > 1.0 and ql <= 1.0                     # (14b) on successive evaluations, recursive one decreasing
        ccrit = qc >= 1.0                                  # (14c)
        margin_b = min(qt - 1.0, 1.0 - ql) if bcrit else max(1.0 - qt if qt <= 1.0 else 0.0, ql - 1.0 if ql > 1.0 else 0.0)
        margin = min(margin, margin_a, margin_b, abs(qc - 1.0))
        mask = (1 if a else 0) | (2 if bcrit else 0) | (4 if ccrit else 0)
        if mask:
            return k, mask, margin, drift / true
        t_prev, l_prev = true, low
    return None, 0, margin, 0.0
