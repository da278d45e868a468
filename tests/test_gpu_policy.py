"""Row a5 on the device: every branch of the stage-switch policy as an EXACT expectation.

  * test_device_policy_truth_table: the decision function the solver kernels run (csrc/cuth_policy.cuh, through the
    cuth_policy_probe hook) on hand-picked norms either side of each printed constant -- the expectations are typed
    here from eq. (14a)-(14c), not taken from oracle/policy.py;
  * whole solves in which (14a)+soft restart, (14c)+hard, (14b)+hard, (14b)+soft, (14a)+(14c) together, and the
    late-stage hard restart are each the expected outcome, with the switch iteration derived by tests/policy_scan.py
    from a plain PCG history (no policy code); run in every home of the loop that has the operator: CUDA graph (flat
    and z-marching / fused), persistent kernel, cluster-resident kernel, batched kernel.
Mutation check (done by hand on the device code, 2026-11): 0.25 -> 0.49 in switch_criteria (14c), 0.81 -> 0.9025 in
(14b), sw2 = rtol -> rtol^(2/3), soft_drift2 1e-2 -> 0.49, or testing (14c) before (14b) when forming `reason`, each
fail test_device_policy_truth_table and at least one scenario test."""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O
from oracle import policy as P
from gpu_util import grid_from_workload, to_dev
from policy_scan import expected_switch

pytestmark = pytest.mark.gpu

HOMES = ["flat-graph", "persistent", "cluster", "cluster-smem", "zmarch-graph", "zmarch-k1x1", "batch", "batch-cluster",
         "batch-cluster-smem"]


def _solve(w, b, home, precision, rtol=1e-8, period=20, max_iters=200000):
    """One solve through the C ABI in the given home of the loop; returns (x, Result)."""
    import torch
    import paper_2606_17850_b200 as cu
    tune = {"flat-graph": cu.Tuning(traversal=1, loop_mode=1), "persistent": cu.Tuning(traversal=1, loop_mode=2),
            "cluster": cu.Tuning(loop_mode=3),                     # rows in registers where they fit (cuth_cluster_reg.cuh)
            "cluster-smem": cu.Tuning(loop_mode=4),                # rows in shared memory (cuth_cluster.cuh)
            "zmarch-graph": cu.Tuning(traversal=2, k1_variant=2), "zmarch-k1x1": cu.Tuning(traversal=2, k1_variant=1),
            "batch": cu.Tuning(loop_mode=2), "batch-cluster": cu.Tuning(loop_mode=3),
            "batch-cluster-smem": cu.Tuning(loop_mode=4)}[home]
    opts = cu.Opts(precision=precision, rtol=rtol, max_iters=max_iters, true_resid_period=period, tuning=tune)
    M = cu.DiaMatrix(grid_from_workload(w))
    if home.startswith("batch"):
        S = cu.BatchSolver(M, 2, opts)
        X = torch.zeros(2, w.n, dtype=torch.float64, device="cuda")
        S.solve(torch.stack([to_dev(b), to_dev(0.5 * b)]), X)
        rs = S.results()
        # the second system is the first one scaled: the same decisions (every criterion is scale-free)
        assert (rs[1].switch_reason, rs[1].switch_mask, rs[1].hard_restarts, rs[1].soft_restarts) == \
               (rs[0].switch_reason, rs[0].switch_mask, rs[0].hard_restarts, rs[0].soft_restarts)
        return X[0].cpu().numpy(), rs[0]
    S = cu.Solver(M, opts)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    S.solve(to_dev(b), x)
    r = S.result()
    S.close()
    return x.cpu().numpy(), r


def _rel(A, b, x):
    return np.linalg.norm(b - O.spmv(A, x)) / np.linalg.norm(b)


# ---------------------------------------------------------------- the decision function, scalar by scalar
def test_device_policy_truth_table():
    import paper_2606_17850_b200 as cu
    q = cu.cuth_policy_probe
    bb, rtol = 1.0, 1e-8                       # tol^2 = 1e-16, (14a): ||r_low||^2 <= 1e-8
    sq = lambda v: v * v

    def early(low, true, drift, true_prev=1.0, low_prev=1.0, **kw):
        return q(sq(low), sq(true), sq(drift), sq(true_prev), sq(low_prev), bb, rtol, **kw)

    # nothing holds: stay early, no restart
    r = early(0.5, 0.5, 0.01)
    assert (r["go"], r["stage"], r["switch_mask"], r["switch_reason"], r["restart"], r["promotions"]) == (1, 0, 0, 0, 0, 0)
    # (14a) PAPER.md:384: ||r_low|| <= sqrt(1e-8) = 1e-4, either side
    assert early(0.99e-4, 0.99e-4, 1e-6, 1e-3, 1e-3)["switch_mask"] == 1
    assert early(1.01e-4, 1.01e-4, 1e-6, 1e-3, 1e-3)["switch_mask"] == 0
    # (14b) PAPER.md:387 + :400: true > 0.9 true_prev while low <= 0.9 low_prev
    assert early(0.89, 0.91, 0.05)["switch_mask"] == 2
    assert early(0.89, 0.89, 0.05)["switch_mask"] == 0          # the true residual did drop by > 10 %
    assert early(0.91, 0.91, 0.05)["switch_mask"] == 0          # the recursive one did not decrease (R-G9)
    assert early(9.0, 9.0, 0.05)["switch_mask"] == 0            # both rise together: CG's residual is not monotone
    # (14c) PAPER.md:392: ||r_true - r_low|| >= 0.5 ||r_true||
    assert early(0.3, 0.5, 0.251)["switch_mask"] == 4
    assert early(0.3, 0.5, 0.249)["switch_mask"] == 0
    # several at once: all bits, reason = the first in the printed order
    r = early(0.3, 0.95, 0.8)
    assert (r["switch_mask"], r["switch_reason"]) == (6, 2)
    r = early(0.5e-4, 2e-4, 1.6e-4, 1e-3, 1e-3)
    assert (r["switch_mask"], r["switch_reason"]) == (5, 1)
    r = early(0.5e-4, 0.95e-3, 0.9e-3, 1e-3, 1e-3)
    assert (r["switch_mask"], r["switch_reason"]) == (7, 1)
    # the switch itself: stage -> late, one promotion; restart kind by the drift (R-G11: soft while <= 0.1 ||r_true||)
    r = early(0.99e-4, 0.99e-4, 0.09 * 0.99e-4, 1e-3, 1e-3)
    assert (r["stage"], r["promotions"], r["restart"], r["go"]) == (1, 1, 2, 1)
    r = early(0.99e-4, 0.99e-4, 0.11 * 0.99e-4, 1e-3, 1e-3)
    assert (r["stage"], r["promotions"], r["restart"]) == (1, 1, 1)
    assert early(0.3, 0.5, 0.3)["restart"] == 1                 # (14c) always means a large drift: p = z
    assert early(0.89, 0.91, 0.05, soft_drift=-1.0)["restart"] == 1     # soft restart disabled
    # stopping rule first (R-G7): a verified true residual ends the solve, no switch
    r = early(0.9e-8, 0.9e-8, 1e-10, 1e-3, 1e-3, conv_rec=True)
    assert (r["go"], r["status"], r["switch_mask"], r["stage"]) == (0, 0, 0, 0)
    # early stage, recursive residual passed but the true one did not: that IS (14a)
    r = early(0.9e-8, 2e-8, 1.5e-8, 1e-3, 1e-3, conv_rec=True)
    assert (r["go"], r["switch_reason"], r["switch_mask"] & 1, r["restart"]) == (1, 1, 1, 1)
    # late stage: failed verification -> hard restart; a periodic look without conv_rec -> nothing
    r = q(sq(0.9e-8), sq(2e-8), sq(1.5e-8), 1.0, 1.0, bb, rtol, late=True, conv_rec=True)
    assert (r["go"], r["stage"], r["restart"], r["switch_mask"], r["promotions"]) == (1, 1, 1, 0, 0)
    r = q(sq(0.5), sq(0.5), sq(0.4), 1.0, 1.0, bb, rtol, late=True)
    assert (r["go"], r["restart"], r["switch_mask"]) == (1, 0, 0)
    # iteration cap
    r = early(0.5, 0.5, 0.01, capped=True)
    assert (r["go"], r["status"]) == (0, 1)
    # rtol >= 1: the stopping threshold itself bounds (14a) from below
    r = q(sq(1.5), sq(2.5), sq(0.1), sq(10.0), sq(10.0), 1.0, 2.0, conv_rec=True)
    assert (r["go"], r["switch_mask"] & 1, r["switch_reason"]) == (1, 1, 1)


# ---------------------------------------------------------------- (14a) + soft restart: the product path
@pytest.mark.parametrize("home", HOMES)
def test_14a_with_soft_restart(home):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    ref = O.pcg(A, w.power, rtol=1e-8, hist_len=2000)
    first = int(np.argmax(ref.hist[:ref.iterations + 1] <= 1e-4))     # first iteration with ||r|| <= sqrt(rtol) ||b||
    x, r = _solve(w, w.power, home, cu.MIXED)
    assert r.status == 0 and _rel(A, w.power, x) <= 1e-8
    assert (r.promotions, r.switch_reason, r.switch_mask) == (1, 1, 1)
    assert (r.soft_restarts, r.hard_restarts) == (1, 0)
    assert abs(r.switch_iteration - first) <= 2
    assert abs(r.iterations - ref.iterations) <= 3                    # a soft restart costs nothing (R-G11)


# ---------------------------------------------------------------- (14c) + hard restart: the paper's A2 literally
@pytest.mark.parametrize("home", ["flat-graph", "persistent"])
@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=1, nx=12, ny=10, nz=8, n_hot=2)])
def test_14c_with_hard_restart_standard_form(home, kw):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    k, mask, margin, drift = expected_switch(A, P.standard_form_fp32_operator(A), w.power, 1e-8, 20, 400)
    assert mask == 4 and margin >= 0.05
    x, r = _solve(w, w.power, home, cu.MIXED_STD32)
    assert r.status == 0 and _rel(A, w.power, x) <= 1e-8
    assert (r.promotions, r.switch_reason, r.switch_mask, r.switch_iteration) == (1, 3, 4, k)
    assert (r.soft_restarts, r.hard_restarts) == (0, 1)
    ref = O.pcg(A, w.power, rtol=1e-8)
    assert np.abs(x - ref.x).max() <= 1e-4                             # the policy rescues the literal A2 as well
    assert r.iterations > ref.iterations + 20                          # ... at the price of the hard restart


# ---------------------------------------------------------------- (14b)
@pytest.mark.parametrize("home", ["flat-graph", "persistent"])
def test_14b_with_hard_restart(home):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(6, nx=45, ny=38, nz=10, n_hot=6)
    A = O.assemble_workload(w)
    k, mask, margin, drift = expected_switch(A, P.standard_form_fp32_operator(A), w.power, 1e-8, 5, 600)
    assert mask == 2 and margin >= 3e-3 and 0.1 < drift < 0.5
    x, r = _solve(w, w.power, home, cu.MIXED_STD32, period=5)
    assert r.status == 0 and _rel(A, w.power, x) <= 1e-8
    assert (r.promotions, r.switch_reason, r.switch_mask, r.switch_iteration) == (1, 2, 2, k)
    assert (r.soft_restarts, r.hard_restarts) == (0, 1)


@pytest.mark.parametrize("home", ["flat-graph", "persistent"])
def test_14b_with_soft_restart(home):
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    k, mask, margin, drift = expected_switch(A, P.standard_form_fp32_operator(A), w.power, 1e-8, 1, 400)
    assert mask == 2 and drift < 0.1 and margin >= 5e-4
    x, r = _solve(w, w.power, home, cu.MIXED_STD32, period=1)
    assert r.status == 0 and _rel(A, w.power, x) <= 1e-8
    assert (r.switch_reason, r.switch_mask, r.switch_iteration) == (2, 2, k)
    assert (r.soft_restarts, r.hard_restarts) == (1, 0)


# ---------------------------------------------------------------- (14a) and (14c) together; late-stage restarts
@pytest.mark.parametrize("home", HOMES)
def test_14a_and_14c_together_then_late_stage_hard_restarts(home):
    """rtol = 1e-15: (14a)'s threshold 3e-8 ||b|| lies below the ~5e-8 floor of the difference-form operator, so
    when the recursive residual gets there the drift is already > 0.5 ||r_true||: both bits, reason 1.  1e-15 is not
    reachable in fp64: the solve ends at the cap after several late-stage verification failures (hard restarts)."""
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    s = np.zeros((w.nz, w.nx * w.ny))
    s[w.nz - 1] += w.h_top * w.dx * w.dy
    k, mask, margin, drift = expected_switch(A, P.early_stage_operator(A, s.reshape(-1)), w.power, 1e-15, 20, 400)
    assert mask == 5 and margin >= 0.01
    x, r = _solve(w, w.power, home, cu.MIXED, rtol=1e-15, max_iters=1500)
    assert (r.switch_reason, r.switch_mask, r.switch_iteration) == (1, 5, k)
    assert r.status == 1 and r.iterations == 1500
    assert r.soft_restarts == 0 and r.hard_restarts >= 2
    assert r.true_resid_evals >= r.hard_restarts + 1
    assert _rel(A, w.power, x) <= 1e-9                                  # still a far better x than rtol 1e-8 asks for


@pytest.mark.parametrize("home", HOMES)
@pytest.mark.parametrize("kw", [dict(cfg=1), dict(cfg=6, nx=20, ny=18, nz=10, n_hot=3)])
def test_late_stage_verification_failure_is_a_hard_restart(home, kw):
    """FP64 mode, rtol = 1e-10: the recursive residual passes while b - A x does not; r := b - A x, p := z, continue --
    exactly what oracle_pcg does (same iteration count to within summation order)."""
    import paper_2606_17850_b200 as cu
    w = W.make_workload(**kw)
    A = O.assemble_workload(w)
    ref = O.pcg(A, w.power, rtol=1e-10)
    x, r = _solve(w, w.power, home, cu.FP64, rtol=1e-10)
    assert r.status == 0 and _rel(A, w.power, x) <= 1e-10
    assert (r.promotions, r.switch_reason, r.switch_mask, r.soft_restarts) == (0, 0, 0, 0)
    assert r.hard_restarts >= 1 and r.true_resid_evals == r.hard_restarts + 1
    assert abs(r.iterations - ref.iterations) <= max(5, 0.05 * ref.iterations)
    assert np.abs(x - ref.x).max() <= 1e-8 * np.abs(ref.x).max()


def test_standard_form_is_refused_where_it_does_not_exist():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(1, nx=8, ny=6, nz=4, n_hot=1)
    M = cu.DiaMatrix(grid_from_workload(w))
    S = cu.BatchSolver(M, 2, cu.Opts(precision=cu.MIXED_STD32))
    X = torch.zeros(2, w.n, dtype=torch.float64, device="cuda")
    with pytest.raises(cu.CuthError) as e:
        S.solve(torch.ones(2, w.n, dtype=torch.float64, device="cuda"), X)
    assert e.value.code == -3
