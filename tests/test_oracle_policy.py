"""Pins of the step-by-step mixed-precision reference (oracle/policy.py), CPU only.

Every branch of the stage-switch policy of PAPER.md §IV-D is the EXPECTED outcome of at
least one test, and the expectation never comes from pcg_mixed itself:
  * eq. (14a)-(14c) as truth tables on hand-picked norms either side of the printed constants (0.9, 0.5,
    sqrt(eps));
  * whole solves whose switch iteration / criterion are derived by tests/policy_scan.py from the residual history
    of a plain PCG on the early-stage operator (no policy code involved);
  * mathematical facts: the converged x is A^-1 b (direct solve / Cholesky); a soft restart with zero drift is a
    no-op (same iterates as plain PCG); the late-stage verification failure behaves exactly like oracle_pcg.
Mutation check (done by hand, 2026-11): changing 0.5 -> 0.7 in crit_14c, 0.9 -> 0.95 in crit_14b, sqrt -> cbrt
in crit_14a or soft_drift 0.1 -> 0.7 in restart_kind fails test_criteria_truth_table /
test_restart_kind_truth_table AND at least one scenario test below; swapping the order of (14b) and (14c) in
first_reason fails test_first_reason_follows_the_printed_order."""
import numpy as np
import pytest
import scipy.linalg as sla

import workloads as W
from oracle import oracle as O
from oracle import policy as P
from direct_solve import solve_layered
from policy_scan import expected_switch


def row_sums(w):
    s = np.zeros((w.nz, w.nx * w.ny))
    s[w.nz - 1] += w.h_top * w.dx * w.dy
    if w.transient:
        s += (w.cvol * (w.dx * w.dy * w.dz) / w.dt)[:, None]
    return s.reshape(-1)


# ---------------------------------------------------------------- eq. (14a)-(14c) as truth tables
def test_criteria_truth_table():
    # (14a): eps = 1e-8 -> n = -4: ||r_low|| <= 1e-4 (x ||b||)
    assert P.crit_14a(0.99e-4, 1e-8, 1.0) and P.crit_14a(1e-4, 1e-8, 1.0) and not P.crit_14a(1.01e-4, 1e-8, 1.0)
    assert P.crit_14a(2.9e-3, 1e-6, 3.0) and not P.crit_14a(3.1e-3, 1e-6, 3.0)       # relative to ||b|| = 3
    assert P.crit_14a(0.99e-6, 1e-12, 1.0) and not P.crit_14a(1.01e-6, 1e-12, 1.0)
    # (14b): true residual > 0.9 x previous although the recursive one fell to <= 0.9 x previous
    assert P.crit_14b(0.91, 1.0, 0.89, 1.0)
    assert not P.crit_14b(0.89, 1.0, 0.89, 1.0)        # the true residual did drop by more than 10 %
    assert not P.crit_14b(0.91, 1.0, 0.91, 1.0)        # the recursive one did not decrease: no verdict (R-G9)
    assert P.crit_14b(1.5, 1.0, 0.5, 1.0)              # true residual rising while the recursive one halves
    assert not P.crit_14b(9.0, 1.0, 9.0, 1.0)          # both rise together (CG's residual is not monotone)
    assert P.crit_14b(2 * 0.91, 2.0, 3 * 0.9, 3.0)     # scale-free
    # (14c)
    assert P.crit_14c(0.5, 1.0) and P.crit_14c(0.51, 1.0) and not P.crit_14c(0.49, 1.0)
    assert P.crit_14c(1.0, 2.0) and not P.crit_14c(0.98, 2.0)


def test_switch_mask_and_first_reason_follow_the_printed_order():
    #                 low   true  drift  true_prev low_prev  eps   ||b||
    none = P.switch_mask(0.5, 0.5, 0.01, 1.0, 1.0, 1e-8, 1.0)
    a = P.switch_mask(0.9e-4, 0.9e-4, 1e-6, 1e-3, 1e-3, 1e-8, 1.0)
    b = P.switch_mask(0.6, 0.95, 0.40, 1.0, 1.0, 1e-8, 1.0)
    c = P.switch_mask(0.3, 0.5, 0.30, 1.0, 1.0, 1e-8, 1.0)
    bc = P.switch_mask(0.3, 0.95, 0.80, 1.0, 1.0, 1e-8, 1.0)
    ac = P.switch_mask(0.5e-4, 2e-4, 1.6e-4, 1e-3, 1e-3, 1e-8, 1.0)
    abc = P.switch_mask(0.5e-4, 0.95e-3, 0.9e-3, 1e-3, 1e-3, 1e-8, 1.0)
    assert (none, a, b, c, bc, ac, abc) == (0, 1, 2, 4, 6, 5, 7)
    assert [P.first_reason(m) for m in (0, 1, 2, 4, 6, 5, 7, 3)] == [0, 1, 2, 3, 2, 1, 1, 1]


def test_restart_kind_truth_table():
    # PAPER.md:402 / R-G11: soft (2) while ||r_true - r_low|| <= 0.1 ||r_true||, hard (1) beyond
    assert P.restart_kind(0.05, 1.0, 0.1) == 2 and P.restart_kind(0.1, 1.0, 0.1) == 2
    assert P.restart_kind(0.11, 1.0, 0.1) == 1 and P.restart_kind(0.6, 1.0, 0.1) == 1
    assert P.restart_kind(0.0, 1.0, -1.0) == 1         # soft restart disabled


# ---------------------------------------------------------------- early-stage operators
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


def test_standard_form_operator_is_the_fp32_rounding_of_every_entry():
    w = W.make_workload(1, nx=6, ny=5, nz=4, n_hot=1)
    A = O.assemble_workload(w)
    S = P.standard_form_fp32_operator(A)
    assert np.array_equal(S.val, A.val.astype(np.float32).astype(np.float64))
    assert np.array_equal(S.col, A.col) and np.array_equal(S.rowptr, A.rowptr)
    # F2: rounding D0 destroys the row sums -- A2 . 1 is off by ~ulp32(D0) ~ 1e-11 W/K, i.e. by more than
    # a thousandth of the whole convective term h dx dy = 1e-8 W/K that fixes the mean temperature
    dev = np.abs(O.spmv(S, np.ones(w.n)) - row_sums(w)).max()
    assert dev > 1e-3 * w.h_top * w.dx * w.dy


# ---------------------------------------------------------------- (14a) + soft restart: the ordinary case
@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=2, nx=40, ny=36, nz=16, n_hot=6)])
def test_mixed_reference_converges_to_the_direct_solution(kw):
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, period=20)
    assert res.status == 0 and res.rel_resid_true <= 1e-8
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    assert np.abs(res.x - xd).max() <= 1e-4
    assert np.linalg.norm(w.power - O.spmv(A, res.x)) <= 1e-8 * np.linalg.norm(w.power)
    assert res.promotions == 1 and res.switch_reason == 1 and res.switch_mask == P.CRIT_A   # (14a) alone
    assert (res.soft_restarts, res.hard_restarts) == (1, 0)
    ref = O.pcg(A, w.power, rtol=1e-8, hist_len=5000)
    first = int(np.argmax(ref.hist[:ref.iterations + 1] <= 1e-4))         # first iteration with ||r|| <= sqrt(rtol) ||b||
    assert abs(res.switch_iteration - first) <= 2
    assert abs(res.iterations - ref.iterations) <= max(3, 0.03 * ref.iterations)   # soft restart: no penalty


def test_soft_restart_with_zero_drift_is_a_no_op_and_a_hard_one_costs_iterations():
    """R-G11: Alg. 1 line 12 with beta = rho(r_true) / rho_{k-1}.  When r_true == r_low the formula gives back the
    beta of the unswitched iteration, so the switched solve must reproduce plain PCG iterate for iterate.  Early
    operator = A itself makes the drift zero up to rounding."""
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    ref = O.pcg(A, w.power, rtol=1e-8)
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, early_operator=A)
    assert (res.switch_reason, res.soft_restarts, res.hard_restarts) == (1, 1, 0)
    assert res.iterations == ref.iterations
    assert np.abs(res.x - ref.x).max() <= 1e-11 * np.abs(ref.x).max()
    hard = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, early_operator=A, soft_drift=-1.0)
    assert (hard.soft_restarts, hard.hard_restarts) == (0, 1)
    assert hard.iterations >= ref.iterations + 10          # p = z throws the Krylov history away


# ---------------------------------------------------------------- (14c) + hard restart: the paper's A2 literally
@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=1, nx=12, ny=10, nz=8, n_hot=2)])
def test_standard_form_early_stage_switches_by_14c_with_a_hard_restart(kw):
    """with every entry of A2 rounded to fp32 the true residual floors near 1e-2 ||b|| while the
    recursive one keeps falling, so the drift criterion (14c) must fire long before (14a)'s 1e-4 ||b||."""
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    S = P.standard_form_fp32_operator(A)
    k, mask, margin, drift = expected_switch(A, S, w.power, 1e-8, 20, 400)
    assert mask == P.CRIT_C and k % 20 == 0 and margin >= 0.05 and drift >= 0.5
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, period=20, early_operator=S)
    assert res.status == 0 and res.rel_resid_true <= 1e-8
    assert (res.promotions, res.switch_reason, res.switch_mask, res.switch_iteration) == (1, 3, P.CRIT_C, k)
    assert (res.soft_restarts, res.hard_restarts) == (0, 1)               # drift >= 0.5 > 0.1: p = z
    low, true = [e for e in res.evals if e[0] == k][0][1:3]
    assert low > 1e-4 * np.linalg.norm(w.power)                           # (14a) was nowhere near
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    assert np.abs(res.x - xd).max() <= 1e-4


# ---------------------------------------------------------------- (14b): stagnating true residual
def test_stagnating_true_residual_switches_by_14b():
    """cfg-6-like stack, standard-form A2, T = 5: at the switch the recursive residual fell below 0.9 x its previous
    evaluation while the true one did not, and the drift is still < 0.5 ||r_true||: (14b) alone."""
    w = W.make_workload(6, nx=45, ny=38, nz=10, n_hot=6)
    A = O.assemble_workload(w)
    S = P.standard_form_fp32_operator(A)
    k, mask, margin, drift = expected_switch(A, S, w.power, 1e-8, 5, 600)
    assert mask == P.CRIT_B and margin >= 3e-3 and 0.1 < drift < 0.5
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, period=5, early_operator=S)
    assert res.status == 0 and res.rel_resid_true <= 1e-8
    assert (res.promotions, res.switch_reason, res.switch_mask, res.switch_iteration) == (1, 2, P.CRIT_B, k)
    assert (res.soft_restarts, res.hard_restarts) == (0, 1)               # drift > 0.1 ||r_true||


def test_14b_with_a_soft_restart():
    """cfg 1, standard-form A2, T = 1: (14b) fires while the drift is only ~4 % of the true residual, so the restart
    keeps p (kind 2)."""
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    S = P.standard_form_fp32_operator(A)
    k, mask, margin, drift = expected_switch(A, S, w.power, 1e-8, 1, 400)
    assert mask == P.CRIT_B and drift < 0.1 and margin >= 5e-4
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-8, period=1, early_operator=S)
    assert (res.switch_reason, res.switch_mask, res.switch_iteration) == (2, P.CRIT_B, k)
    assert (res.soft_restarts, res.hard_restarts) == (1, 0)
    assert res.status == 0 and res.rel_resid_true <= 1e-8


# ---------------------------------------------------------------- several criteria at once
def test_14a_and_14c_together_below_the_fp32_floor():
    """rtol = 1e-15 puts (14a)'s threshold sqrt(rtol) = 3e-8 below the ~5e-8 floor of the difference-form operator
    (SURVEY F3): when the recursive residual gets there the drift is already large -- both bits, reason = the first
    in the printed order; the solve then runs into max_iters (1e-15 is not reachable in fp64), with late-stage hard
    restarts on the way."""
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    E = P.early_stage_operator(A, row_sums(w))
    k, mask, margin, drift = expected_switch(A, E, w.power, 1e-15, 20, 400)
    assert mask == (P.CRIT_A | P.CRIT_C) and margin >= 0.01
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-15, period=20, max_iters=1500)
    assert (res.switch_reason, res.switch_mask, res.switch_iteration) == (1, P.CRIT_A | P.CRIT_C, k)
    assert res.status == 1 and res.iterations == 1500
    assert res.hard_restarts >= 2 and res.soft_restarts == 0


# ---------------------------------------------------------------- late stage: failed verification
@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=6, nx=20, ny=18, nz=10, n_hot=3)])
def test_late_stage_verification_failure_is_a_hard_restart_like_oracle_pcg(kw):
    """R-G7: at rtol = 1e-10 the recursive residual passes the test while b - A x does not (drift of ~1e-10 ||b||
    after a few hundred fp64 iterations): r := b - A x, p := z, continue -- the rule oracle_pcg (C++) implements on
    its own; same iteration count, same x."""
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    ref = O.pcg(A, w.power, rtol=1e-10)
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-10, start_early=False)
    assert res.status == 0 and ref.status == 0
    assert res.promotions == 0 and res.switch_reason == 0
    assert res.hard_restarts >= 1 and res.soft_restarts == 0 and res.true_resid_evals == res.hard_restarts + 1
    assert res.iterations == ref.iterations
    assert np.abs(res.x - ref.x).max() <= 1e-10 * np.abs(ref.x).max()


def test_mixed_reference_tiny_vs_cholesky_and_zero_rhs():
    w = W.make_workload(1, nx=6, ny=5, nz=4, n_hot=1)
    A = O.assemble_workload(w)
    xs = sla.cho_solve(sla.cho_factor(A.to_scipy().toarray()), w.power)
    res = P.pcg_mixed(A, row_sums(w), w.power, rtol=1e-9, period=5)
    assert res.status == 0 and np.abs(res.x - xs).max() <= 1e-6 * np.abs(xs).max()
    z = P.pcg_mixed(A, row_sums(w), np.zeros(w.n), x0=np.ones(w.n))
    assert z.status == 0 and z.iterations == 0 and np.all(z.x == 0)
