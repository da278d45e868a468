// cuth_policy.cuh -- the scalar side of the PCG loop: what happens to the control block after each
// grid-wide reduction (Alg. 1 lines 7, 11, 13; stopping rule R-G7; stage switch eq. (14a)-(14c),
// PAPER.md:382-402).  One copy of the logic, used by the last-CTA epilogues of the graph path (Ctl in
// global memory) and by every CTA of the persistent path (Ctl replicated in shared memory).
#pragma once
#include "cuth_internal.cuh"

namespace cuth {

// What the matrix object says about itself (header words written by the builder / the importers, device memory):
// 0 = usable for this call, else the CUTH_SOLVE_* status that ends the solve before it starts.
__device__ __forceinline__ int matrix_refusal(const Ctx& c) {
  const unsigned long long* h = c.A.hdr;
  if (h[kHdrMagic] != kMagic || (int64_t)h[kHdrNx] != c.A.nx || (int64_t)h[kHdrNy] != (int64_t)c.A.ny ||
      (int64_t)h[kHdrNz] != (int64_t)c.A.nz)
    return CUTH_SOLVE_BAD_MATRIX;
  if (c.transient_call && (h[kHdrTransient] == 0ull || h[kHdrImported] != 0ull)) return CUTH_SOLVE_NOT_TRANSIENT;
  if (c.precision == CUTH_MIXED && h[kHdrMixedOk] == 0ull) return CUTH_SOLVE_FP64_ONLY;
  return 0;
}

// After r0 = b - A1 x0: sums rho = r.z, rr = r.r, bb = b.b.  Returns 1 if the loop must run.
__device__ __forceinline__ unsigned policy_init(Ctl* ctl, const Ctx& c, double rho, double rr, double bb) {
  ctl->rho = rho; ctl->rr = rr; ctl->bb = bb;
  ctl->tol2 = c.rtol * c.rtol * bb;
  // (sqrt(rtol) ||b||)^2, eq. (14a) relative (R-G8); never below the stopping threshold itself (rtol >= 1), so
  // that a recursive residual that passes the stopping test always satisfies (14a)
  ctl->sw2 = fmax(c.rtol, c.rtol * c.rtol) * bb;
  ctl->beta = 0.0; ctl->alpha = 0.0;
  ctl->tt = rr; ctl->tt_prev = rr; ctl->rr_prev_eval = rr;
  ctl->stage = (c.precision == CUTH_MIXED || c.precision == CUTH_MIXED_STD32) ? 0 : 1;
  ctl->beta_zero = 1;                            // Chebyshev path: the first p is z (Alg. 1 line 3)
  unsigned go = 1u;
  const int refusal = matrix_refusal(c);
  if (refusal) { ctl->status = refusal; ctl->refused = 1; go = 0u; }
  else if (bb == 0.0) { ctl->zero_rhs = 1; ctl->status = CUTH_SOLVE_CONVERGED; ctl->tt = 0.0; ctl->rr = 0.0; go = 0u; }
  else if (rr <= ctl->tol2) { ctl->status = CUTH_SOLVE_CONVERGED; go = 0u; }          // r0 IS the true residual
  else if (!(rho == rho) || !(rr == rr)) { ctl->status = CUTH_SOLVE_BREAKDOWN; go = 0u; }
  return go;
}

// After mu = A p: Alg. 1 line 7.  defer_x (fused path): x += alpha p is left to the NEXT K1, which has p in registers
// anyway -- unless this iteration is certain to end in a true-residual evaluation (period reached in the early stage,
// or the iteration cap): then K2 applies it at once (ctl->xnow), k_flush_x finds nothing pending and the next K1,
// seeing xalpha = 0, neither reads nor writes x.  Same fma on the same operands either way: identical iterates.
__device__ __forceinline__ void policy_after_spmv(Ctl* ctl, double pAp, bool defer_x, const Ctx* c = nullptr) {
  ctl->pAp = pAp;
  const double rho = ctl->rho;
  ctl->xnow = 0;
  if (!(pAp > 0.0) || !(pAp <= 1.79e308) || !(rho == rho)) {
    ctl->alpha = 0.0; ctl->xalpha = 0.0;
    ctl->status = CUTH_SOLVE_BREAKDOWN;
  } else {
    const double alpha = rho / pAp;
    ctl->alpha = alpha;
    if (defer_x) {
      const bool now = c && !ctl->no_graph &&
                       ((ctl->stage == 0 && ctl->since_eval + 1 >= c->period) || ctl->it + 1 >= c->max_iters);
      ctl->xnow = now ? 1 : 0;
      ctl->xalpha = now ? 0.0 : alpha;
    }
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
  ctl->halt = ((!go || want) && !ctl->no_graph) ? 1 : 0;      // replays outside the graph never halt
}

// Eq. (14a)-(14c) on SQUARED norms -- the grid-wide sums the kernels produce -- so the printed
// constants appear squared: 0.9^2 = 0.81, 0.5^2 = 0.25.  Bit 0 = (14a), bit 1 = (14b), bit 2 = (14c).
//   (14a)  ||r_low||^2 <= rtol ||b||^2                  (relative form of 10^(log10(eps)/2), R-G8; sw2)
//   (14b)  ||r_true||^2 > 0.81 ||r_true,prev||^2  while  ||r_low||^2 <= 0.81 ||r_low,prev||^2   (successive
//          evaluations; "despite a decreasing recursive one", R-G9)
//   (14c)  ||r_true - r_low||^2 >= 0.25 ||r_true||^2     (second print, R-G10)
__device__ __forceinline__ int switch_criteria(double rr, double tt, double dd, double tt_prev, double rr_prev,
                                               double sw2) {
  int mask = 0;
  if (rr <= sw2) mask |= 1;
  if (tt > 0.81 * tt_prev && rr <= 0.81 * rr_prev) mask |= 2;
  if (dd >= 0.25 * tt) mask |= 4;
  return mask;
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
    // "triggered when any of the following holds"; the reason reported is the first in the
    // printed order.  A recursive residual that passed the stopping test satisfies (14a) by construction of sw2.
    const int mask = switch_criteria(rr, tt, dd, ctl->tt_prev, ctl->rr_prev_eval, ctl->sw2);
    if (mask) {
      const int reason = (mask & 1) ? 1 : ((mask & 2) ? 2 : 3);
      ctl->stage = 1; ctl->promotions += 1; ctl->switch_reason = reason; ctl->switch_mask = mask; ctl->switch_it = ctl->it;
      // hot restart.  Small drift: r is recomputed, p keeps its history through its
      // defining equation p = z + beta p ("preserving the established Krylov subspace");
      // large drift ((14c)): the direction is rebuilt from scratch, p = z.
      restart = (c.soft_restart && dd <= c.soft_drift2 * tt) ? 2 : 1;
    }
  }
  ctl->tt_prev = tt;
  ctl->rr_prev_eval = rr;
  ctl->restart = restart;
  if (restart == 1) ctl->hard_restarts += 1;
  else if (restart == 2) ctl->soft_restarts += 1;
  ctl->halt = go ? 0 : 1;
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
  res.switch_mask = ctl->switch_mask;
  res.hard_restarts = ctl->hard_restarts;
  res.soft_restarts = ctl->soft_restarts;
  res.reserved = 0;
  *c.result = res;
}

}  // namespace cuth
