// cuth_policy.cuh -- the scalar side of the PCG loop: what happens to the control block after each
// grid-wide reduction (Alg. 1 lines 7, 11, 13; stopping rule R-G7; stage switch eq. (14a)-(14c),
// PAPER.md:382-402).  One copy of the logic, used by the last-CTA epilogues of the graph path (Ctl in
// global memory) and by every CTA of the persistent path (Ctl replicated in shared memory).
#pragma once
#include "cuth_internal.cuh"

namespace cuth {

// After r0 = b - A1 x0: sums rho = r.z, rr = r.r, bb = b.b.  Returns 1 if the loop must run.
__device__ __forceinline__ unsigned policy_init(Ctl* ctl, const Ctx& c, double rho, double rr, double bb) {
  ctl->rho = rho; ctl->rr = rr; ctl->bb = bb;
  ctl->tol2 = c.rtol * c.rtol * bb;
  ctl->sw2 = c.rtol * bb;                        // (sqrt(rtol) ||b||)^2, eq. (14a) relative (R-G8)
  ctl->beta = 0.0; ctl->alpha = 0.0;
  ctl->tt = rr; ctl->tt_prev = rr; ctl->rr_prev_eval = rr;
  ctl->stage = (c.precision == CUTH_MIXED) ? 0 : 1;
  ctl->beta_zero = 1;                            // Chebyshev path: the first p is z (Alg. 1 line 3)
  unsigned go = 1u;
  if (bb == 0.0) { ctl->zero_rhs = 1; ctl->status = CUTH_SOLVE_CONVERGED; ctl->tt = 0.0; ctl->rr = 0.0; go = 0u; }
  else if (rr <= ctl->tol2) { ctl->status = CUTH_SOLVE_CONVERGED; go = 0u; }          // r0 IS the true residual
  else if (!(rho == rho) || !(rr == rr)) { ctl->status = CUTH_SOLVE_BREAKDOWN; go = 0u; }
  return go;
}

// After mu = A p: Alg. 1 line 7.
__device__ __forceinline__ void policy_after_spmv(Ctl* ctl, double pAp, bool defer_x) {
  ctl->pAp = pAp;
  const double rho = ctl->rho;
  if (!(pAp > 0.0) || !(pAp <= 1.79e308) || !(rho == rho)) {
    ctl->alpha = 0.0; ctl->xalpha = 0.0;
    ctl->status = CUTH_SOLVE_BREAKDOWN;
  } else {
    const double alpha = rho / pAp;
    ctl->alpha = alpha;
    if (defer_x) ctl->xalpha = alpha;            // fused path: x += alpha p is applied by the next K1
  }
}

// After r -= alpha mu: rho_new = r.z, rr = r.r.  Alg. 1 lines 11, 13 and the "evaluate the true residual
// now?" decision.  go: keep looping; want: run the true-residual branch in this pass.
__device__ __forceinline__ void policy_after_update(Ctl* ctl, const Ctx& c, double rho_new, double rr,
                                                    unsigned& go, unsigned& want) {
  go = 1u; want = 0u;
  if (ctl->status == CUTH_SOLVE_BREAKDOWN) {
    go = 0u;
  } else {
    if (!c.cheb) {                               // Chebyshev: rho and beta come from k_cheb_last
      ctl->beta = rho_new / ctl->rho;            // Alg. 1 line 11
      ctl->rho = rho_new;
    }
    ctl->rr = rr;
    const int it = ctl->it + 1;                  // Alg. 1 line 13
    ctl->it = it;
    const int since = ctl->since_eval + 1;
    ctl->since_eval = since;
    const bool conv_rec = rr <= ctl->tol2;
    const bool early = ctl->stage == 0;
    const bool c14a = early && rr <= ctl->sw2;
    const bool periodic = early && since >= c.period;
    const bool capped = it >= c.max_iters;
    const bool bad = !(rr == rr) || (!c.cheb && !(rho_new == rho_new));
    ctl->conv_rec = conv_rec ? 1 : 0;
    if (bad) { ctl->status = CUTH_SOLVE_BREAKDOWN; go = 0u; }
    else if (conv_rec || c14a || periodic || capped) want = 1u;
  }
  ctl->want_true = (int)want;
}

// After t = b - A1 x: tt = ||t||^2, dd = ||t - r||^2.  Stopping rule and eq. (14a)-(14c).  Sets
// ctl->restart (0 none, 1 hard: p = z, 2 soft: p keeps its history).  Returns go.
__device__ __forceinline__ unsigned policy_after_true(Ctl* ctl, const Ctx& c, double tt, double dd) {
  const double rr = ctl->rr;
  ctl->tt = tt; ctl->dd = dd;
  ctl->evals += 1;
  ctl->since_eval = 0;
  ctl->xalpha = 0.0;                             // k_flush_x has just applied it (fused path)
  unsigned go = 1u;
  int restart = 0;
  if (tt <= ctl->tol2) { ctl->status = CUTH_SOLVE_CONVERGED; go = 0u; }
  else if (ctl->it >= c.max_iters) { ctl->status = CUTH_SOLVE_MAX_ITERS; go = 0u; }
  else if (ctl->stage == 1) {
    // late stage: the recursive residual said "converged", the true one disagrees -> replace r,
    // restart the direction (same rule as the oracle), keep iterating.
    if (ctl->conv_rec) restart = 1;
  } else {
    int reason = 0;
    if (ctl->conv_rec) reason = 4;
    else if (rr <= ctl->sw2) reason = 1;                                          // (14a)
    else if (dd >= 0.25 * tt) reason = 3;                                         // (14c): ||t-r|| >= 0.5 ||t||
    else if (tt > 0.81 * ctl->tt_prev && rr <= 0.81 * ctl->rr_prev_eval) reason = 2;     // (14b), R-G9
    if (reason) {
      ctl->stage = 1; ctl->promotions += 1; ctl->switch_reason = reason; ctl->switch_it = ctl->it;
      // hot restart.  Small drift: r is recomputed, p keeps its history through its
      // defining equation p = z + beta p ("preserving the established Krylov subspace");
      // large drift ((14c)): the direction is rebuilt from scratch, p = z.
      restart = (c.soft_restart && dd <= c.soft_drift2 * tt) ? 2 : 1;
    }
  }
  ctl->tt_prev = tt;
  ctl->rr_prev_eval = rr;
  ctl->restart = restart;
  return go;
}

// After r := t: rho = r.z, rr = r.r of the replaced residual.
__device__ __forceinline__ void policy_after_restart(Ctl* ctl, const Ctx& c, int mode, double rho, double rr) {
  // mode 1: beta = 0 => p = z.  mode 2: beta_k = rho(new r) / rho_k, with rho_k = rho_rec / beta_rec.
  if (c.cheb) {        // the next k_cheb_last forms rho(new r) and beta = rho_new / rho_k itself
    ctl->beta_zero = (mode == 1) ? 1 : 0;
  } else {
    ctl->beta = (mode == 2 && ctl->rho > 0.0) ? ctl->beta * (rho / ctl->rho) : 0.0;
    ctl->rho = rho;
  }
  ctl->rr = rr; ctl->restart = 0; ctl->conv_rec = 0;
}

__device__ __forceinline__ void write_result(const Ctl* ctl, const Ctx& c) {
  cuth_result_t res;
  res.status = ctl->status == CUTH_SOLVE_RUNNING ? CUTH_SOLVE_MAX_ITERS : ctl->status;
  res.iterations = ctl->it;
  res.promotions = ctl->promotions;
  res.true_resid_evals = ctl->evals;
  const double bb = ctl->bb;
  res.rel_resid_true = bb > 0.0 ? sqrt(ctl->tt / bb) : 0.0;
  res.rel_resid_rec = bb > 0.0 ? sqrt(ctl->rr / bb) : 0.0;
  res.switch_reason = ctl->switch_reason;
  res.switch_iteration = ctl->switch_it;
  *c.result = res;
}

}  // namespace cuth
