// cuth_persistent.cuh -- the whole PCG solve as ONE persistent cooperative kernel, for grids whose
// working set lives in L2 (cfg 1, cfg 2): there a CUDA-graph WHILE iteration costs ~9 us of scheduling
// against a few us of work, so the loop moves inside the kernel and the kernel
// boundaries become grid.sync().  Same arithmetic, same policy code (cuth_policy.cuh) as the graph path:
//   A: p = M^-1 r + beta p                           (Alg. 1 line 12)      grid.sync
//   B: mu = A p, p.mu  -> alpha                      (lines 6-7)           all-reduce (grid.sync inside)
//   C: x += alpha p, r -= alpha mu, r.z, ||r||^2     (lines 8-11, 13)      all-reduce
//   D (when the policy asks): t = b - A1 x, ||t||^2, ||t - r||^2           all-reduce
//   E (restart): r := t, r.z                                               all-reduce
// Every CTA keeps its own copy of the control block in shared memory and takes the same decisions from
// the same sums (each CTA adds the per-CTA partials in the same fixed order), so no scalar ever has to
// be broadcast; CTA 0 writes the result record.  Rows are dealt to threads identically in every
// phase, so only the stencil phases (B, D) need the preceding grid-wide barrier.
#pragma once
#include <cooperative_groups.h>

#include "cuth_kernels.cuh"

namespace cuth {

namespace cg = cooperative_groups;

constexpr int kPersistMaxBlocks = 1024;   // 2 parities x 3 values x 1024 doubles fit the 4 x 8192 partials area

// Sums NV per-thread values over the whole grid; result valid in ALL threads of ALL CTAs.
// partials: [2 parities][3][kPersistMaxBlocks]; phase parity alternates between consecutive calls.
template <int NV>
__device__ __forceinline__ void grid_allreduce(cg::grid_group& grid, double (&v)[NV], double* partials, int& parity,
                                               double* smem /* >= NV*32 + NV */) {
  block_sum<NV>(v, smem);
  double* mine = partials + (size_t)parity * 3 * kPersistMaxBlocks;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) __stcg(&mine[k * kPersistMaxBlocks + blockIdx.x], v[k]);
  }
  grid.sync();
  if (threadIdx.x < 32) {
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      double a = 0.0;
      for (int b = threadIdx.x; b < (int)gridDim.x; b += 32) a += __ldcg(&mine[k * kPersistMaxBlocks + b]);
      a = warp_sum(a);
      if (threadIdx.x == 0) smem[NV * 32 + k] = a;
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = smem[NV * 32 + k];
  __syncthreads();
  parity ^= 1;
}

#define CUTH_ROWS(i_)                                                                            \
  for (int64_t base_ = (int64_t)blockIdx.x * (kThreads * kRows); base_ < n;                      \
       base_ += (int64_t)gridDim.x * (kThreads * kRows))                                         \
    for (int k_ = 0; k_ < kRows; ++k_)                                                           \
      for (int64_t i_ = base_ + threadIdx.x + k_ * kThreads; i_ < n; i_ = n)

__global__ void __launch_bounds__(kThreads, 4) k_pcg_persistent(const Ctx* __restrict__ ctxp, Ctl* ctl_g,
                                                               double* partials) {
  cg::grid_group grid = cg::this_grid();
  __shared__ Ctl sc;
  __shared__ double smem[3 * 32 + 3];
  const Ctx c = *ctxp;
  const int64_t n = c.A.n;
  const bool jac = c.jacobi != 0;
  int parity = 0;
  if (threadIdx.x == 0) sc = *ctl_g;                 // cleared by k_set_ctx
  __syncthreads();

  // ---- Alg. 1 lines 1-3
  {
    double acc[3] = {0.0, 0.0, 0.0};
    CUTH_ROWS(i) {
      const double xi = c.x[i];
      const double bi = c.b[i];
      const double ri = bi - spmv_row<false>(c.A, c.x, i, xi);
      const double zi = jac ? ri * c.A.dinv[i] : ri;
      c.r[i] = ri;
      c.p[i] = 0.0;
      acc[0] = fma(ri, zi, acc[0]); acc[1] = fma(ri, ri, acc[1]); acc[2] = fma(bi, bi, acc[2]);
    }
    grid_allreduce<3>(grid, acc, partials, parity, smem);
    if (threadIdx.x == 0) sc.want_true = (int)policy_init(&sc, c, acc[0], acc[1], acc[2]);   // want_true reused as "go"
    __syncthreads();
  }
  bool go = sc.want_true != 0;

  while (go) {
    // ---- A: p = z + beta p
    {
      const double beta = sc.beta;
      CUTH_ROWS(i) {
        const double ri = c.r[i];
        const double zi = jac ? ri * c.A.dinv[i] : ri;
        c.p[i] = fma(beta, c.p[i], zi);
      }
    }
    grid.sync();
    // ---- B: mu = A p, p.mu
    {
      double acc[1] = {0.0};
      if (sc.stage == 0) {
        CUTH_ROWS(i) { const double pi = c.p[i]; const double m = spmv_row<true>(c.A, c.p, i, pi); c.mu[i] = m; acc[0] = fma(pi, m, acc[0]); }
      } else {
        CUTH_ROWS(i) { const double pi = c.p[i]; const double m = spmv_row<false>(c.A, c.p, i, pi); c.mu[i] = m; acc[0] = fma(pi, m, acc[0]); }
      }
      grid_allreduce<1>(grid, acc, partials, parity, smem);
      if (threadIdx.x == 0) policy_after_spmv(&sc, acc[0], false);
      __syncthreads();
    }
    // ---- C: x, r, dots
    unsigned want = 0u;
    {
      const double alpha = sc.alpha;
      double acc[2] = {0.0, 0.0};
      CUTH_ROWS(i) {
        c.x[i] = fma(alpha, c.p[i], c.x[i]);
        const double ri = fma(-alpha, c.mu[i], c.r[i]);
        const double zi = jac ? ri * c.A.dinv[i] : ri;
        c.r[i] = ri;
        acc[0] = fma(ri, zi, acc[0]); acc[1] = fma(ri, ri, acc[1]);
      }
      grid_allreduce<2>(grid, acc, partials, parity, smem);
      if (threadIdx.x == 0) {
        unsigned g_, w_;
        policy_after_update(&sc, c, acc[0], acc[1], g_, w_);
        sc.exiting = (int)g_;                          // scratch: "go" after this phase
      }
      __syncthreads();
      go = sc.exiting != 0;
      want = (unsigned)sc.want_true;
    }
    if (want) {
      // ---- D: true residual (x is complete: the all-reduce above was a grid-wide barrier)
      double acc[2] = {0.0, 0.0};
      CUTH_ROWS(i) {
        const double ti = c.b[i] - spmv_row<false>(c.A, c.x, i, c.x[i]);
        const double di = ti - c.r[i];
        c.mu[i] = ti;
        acc[0] = fma(ti, ti, acc[0]); acc[1] = fma(di, di, acc[1]);
      }
      grid_allreduce<2>(grid, acc, partials, parity, smem);
      if (threadIdx.x == 0) sc.exiting = (int)policy_after_true(&sc, c, acc[0], acc[1]);
      __syncthreads();
      go = sc.exiting != 0;
      const int mode = sc.restart;
      if (go && mode) {
        // ---- E: r := t
        double a2[2] = {0.0, 0.0};
        CUTH_ROWS(i) {
          const double ri = c.mu[i];
          const double zi = jac ? ri * c.A.dinv[i] : ri;
          c.r[i] = ri;
          a2[0] = fma(ri, zi, a2[0]); a2[1] = fma(ri, ri, a2[1]);
        }
        grid_allreduce<2>(grid, a2, partials, parity, smem);
        if (threadIdx.x == 0) policy_after_restart(&sc, c, mode, a2[0], a2[1]);
        __syncthreads();
      }
    }
  }
  // ---- epilogue
  if (sc.zero_rhs) { CUTH_ROWS(i) c.x[i] = 0.0; }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    sc.exiting = 0;
    write_result(&sc, c);
    *ctl_g = sc;
  }
}

}  // namespace cuth
