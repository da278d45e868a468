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

// Threads per CTA are a launch parameter (the row loops stride by blockDim.x): 256 on grids of up to 64 k rows, 1024
// beyond -- what a grid-wide barrier costs grows with the number of CTAs that take part in it, so the larger grids run
// 128 CTAs of 1024 threads instead of 592 of 256 (cuth_api.cu persistent_config).
constexpr int kPersistMaxThreads = 1024;
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
  {
    // one warp per value: the NV chains of L2 loads run side by side instead of one after the other
    const int lane = threadIdx.x & 31, k = threadIdx.x >> 5;
    if (k < NV) {
      double a = 0.0;
      for (int b = lane; b < (int)gridDim.x; b += 32) a += __ldcg(&mine[k * kPersistMaxBlocks + b]);
      a = warp_sum(a);
      if (lane == 0) smem[NV * 32 + k] = a;
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = smem[NV * 32 + k];
  __syncthreads();
  parity ^= 1;
}

// Rows are dealt to threads with a stride of the whole grid (identically in every phase) and walked two at a
// time: all loads of both rows are issued before the first store, so a phase costs one L2 round trip per pair
// instead of one per row and per store (the stores may alias the loads as far as the compiler knows).
#define CUTH_ROWS2(i0_, i1_, h1_)                                                                \
  for (int64_t i0_ = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, i1_ = i0_ + gstride; i0_ < n;  \
       i0_ += 2 * gstride, i1_ += 2 * gstride)                                                   \
    for (bool h1_ = i1_ < n, once_ = true; once_; once_ = false)

#define CUTH_ROWS(i_)                                                                            \
  for (int64_t i_ = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i_ < n; i_ += gstride)

template <int OP>
__device__ __forceinline__ double persistent_spmv_phase(const Ctx& c, int64_t n, int64_t gstride) {
  double acc = 0.0;
  CUTH_ROWS2(i0, i1, h1) {
    const double p0 = c.p[i0], p1 = h1 ? c.p[i1] : 0.0;
    const double m0 = spmv_row<OP>(c.A, c.p, i0, p0);
    const double m1 = h1 ? spmv_row<OP>(c.A, c.p, i1, p1) : 0.0;
    c.mu[i0] = m0;
    if (h1) c.mu[i1] = m1;
    acc = fma(p0, m0, acc);
    acc = fma(p1, m1, acc);
  }
  return acc;
}

// Phases A and B in one, for the smallest grids (a phase there is one barrier + one L2 round trip): row i forms
// p' = z + beta p not only for itself but also for its six neighbours -- the same fma on the same operands as their
// owners, hence bitwise the same values -- and applies A to them, which removes the barrier between A and B.  p' goes
// to the other direction buffer (the neighbours still read the old one).  21 + 7 independent loads per row instead
// of 3 and 7 + 7: pays only while the barrier outweighs them (measured: 8 k rows 7.26 -> 7.01 us per iteration,
// 66 k rows 8.1 -> 8.9, 1 M rows 23 -> 32), so cuth_api.cu switches it on up to 16 k rows.
template <bool MIXED>
__device__ __forceinline__ double fused_dir_spmv_row(const Ctx& c, const double* __restrict__ pold,
                                                     int64_t i, double beta, bool jac, double& p_i) {
  const DiaDev& A = c.A;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = i + np < n, lo3 = i >= np;
  auto dir = [&](int64_t j) {
    const double rj = c.r[j];
    return fma(beta, pold[j], jac ? rj * A.dinv[j] : rj);
  };
  const double vi = dir(i);
  double acc;
  if (!MIXED) {
    const double a0 = A.d0[i];
    const double a1u = up1 ? A.d1[i] : 0.0, a1l = lo1 ? A.d1[i - 1] : 0.0;
    const double a2u = up2 ? A.d2[i] : 0.0, a2l = lo2 ? A.d2[i - nx] : 0.0;
    const double a3u = up3 ? A.d3[i] : 0.0, a3l = lo3 ? A.d3[i - np] : 0.0;
    const double v1u = up1 ? dir(i + 1) : 0.0, v1l = lo1 ? dir(i - 1) : 0.0;
    const double v2u = up2 ? dir(i + nx) : 0.0, v2l = lo2 ? dir(i - nx) : 0.0;
    const double v3u = up3 ? dir(i + np) : 0.0, v3l = lo3 ? dir(i - np) : 0.0;
    acc = a0 * vi;
    acc = fma(a1u, v1u, acc); acc = fma(a1l, v1l, acc);
    acc = fma(a2u, v2u, acc); acc = fma(a2l, v2l, acc);
    acc = fma(a3u, v3u, acc); acc = fma(a3l, v3l, acc);
  } else {
    const float g1u = up1 ? A.f1[i] : 0.f, g1l = lo1 ? A.f1[i - 1] : 0.f;
    const float g2u = up2 ? A.f2[i] : 0.f, g2l = lo2 ? A.f2[i - nx] : 0.f;
    const float g3u = up3 ? A.f3[i] : 0.f, g3l = lo3 ? A.f3[i - np] : 0.f;
    const double v1u = up1 ? dir(i + 1) : vi, v1l = lo1 ? dir(i - 1) : vi;
    const double v2u = up2 ? dir(i + nx) : vi, v2l = lo2 ? dir(i - nx) : vi;
    const double v3u = up3 ? dir(i + np) : vi, v3l = lo3 ? dir(i - np) : vi;
    const unsigned z = (unsigned)i / (unsigned)np;
    acc = A.s_layer[z] * vi;
    acc = fma((double)g1u, v1u - vi, acc); acc = fma((double)g1l, v1l - vi, acc);
    acc = fma((double)g2u, v2u - vi, acc); acc = fma((double)g2l, v2l - vi, acc);
    acc = fma((double)g3u, v3u - vi, acc); acc = fma((double)g3l, v3l - vi, acc);
  }
  p_i = vi;
  return acc;
}

template <bool MIXED>
__device__ __forceinline__ double persistent_fused_phase(const Ctx& c, const double* __restrict__ pold,
                                                         double* __restrict__ pnew, double beta, bool jac, int64_t n,
                                                         int64_t gstride) {
  double acc = 0.0;
  CUTH_ROWS2(i0, i1, h1) {
    double p0, p1 = 0.0;
    const double m0 = fused_dir_spmv_row<MIXED>(c, pold, i0, beta, jac, p0);
    const double m1 = h1 ? fused_dir_spmv_row<MIXED>(c, pold, i1, beta, jac, p1) : 0.0;
    pnew[i0] = p0; c.mu[i0] = m0;
    if (h1) { pnew[i1] = p1; c.mu[i1] = m1; }
    acc = fma(p0, m0, acc);
    acc = fma(p1, m1, acc);
  }
  return acc;
}

__global__ void __launch_bounds__(kPersistMaxThreads, 1) k_pcg_persistent(const Ctx* __restrict__ ctxp, Ctl* ctl_g,
                                                               double* partials) {
  cg::grid_group grid = cg::this_grid();
  __shared__ Ctl sc;
  __shared__ double smem[3 * 32 + 3];
  const Ctx c = *ctxp;
  const int64_t n = c.A.n;
  const int64_t gstride = (int64_t)gridDim.x * blockDim.x;
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
      const double ri = bi - spmv_row<OP_FP64>(c.A, c.x, i, xi);
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
  const bool fuse = c.persist_fuse != 0;
  double* pcur = c.p;              // the buffer that holds p: the fused phase ping-pongs between c.p and c.p2

  while (go) {
    double acc[1];
    if (fuse) {
      // ---- A + B: p' = z + beta p at the row and its six neighbours, mu = A p', p'.mu
      const double beta = sc.beta;
      double* pnew = (pcur == c.p) ? c.p2 : c.p;
      acc[0] = sc.stage == 0 ? persistent_fused_phase<true>(c, pcur, pnew, beta, jac, n, gstride)
                             : persistent_fused_phase<false>(c, pcur, pnew, beta, jac, n, gstride);
      pcur = pnew;
    } else {
      // ---- A: p = z + beta p
      {
        const double beta = sc.beta;
        CUTH_ROWS2(i0, i1, h1) {
          const double r0 = c.r[i0], q0 = c.p[i0], d0 = jac ? c.A.dinv[i0] : 1.0;
          const double r1 = h1 ? c.r[i1] : 0.0, q1 = h1 ? c.p[i1] : 0.0, d1 = (h1 && jac) ? c.A.dinv[i1] : 1.0;
          c.p[i0] = fma(beta, q0, jac ? r0 * d0 : r0);
          if (h1) c.p[i1] = fma(beta, q1, jac ? r1 * d1 : r1);
        }
      }
      grid.sync();
      // ---- B: mu = A p, p.mu
      acc[0] = sc.stage != 0 ? persistent_spmv_phase<OP_FP64>(c, n, gstride)
                             : (c.early_op == OP_STD32 ? persistent_spmv_phase<OP_STD32>(c, n, gstride)
                                                       : persistent_spmv_phase<OP_DIFF32>(c, n, gstride));
    }
    {
      grid_allreduce<1>(grid, acc, partials, parity, smem);
      if (threadIdx.x == 0) policy_after_spmv(&sc, acc[0], false);
      __syncthreads();
    }
    // ---- C: x, r, dots
    unsigned want = 0u;
    {
      const double alpha = sc.alpha;
      double acc[2] = {0.0, 0.0};
      CUTH_ROWS2(i0, i1, h1) {
        const double x0 = c.x[i0], q0 = pcur[i0], m0 = c.mu[i0], r0 = c.r[i0], d0 = jac ? c.A.dinv[i0] : 1.0;
        double x1 = 0.0, q1 = 0.0, m1 = 0.0, r1 = 0.0, d1 = 1.0;
        if (h1) { x1 = c.x[i1]; q1 = pcur[i1]; m1 = c.mu[i1]; r1 = c.r[i1]; if (jac) d1 = c.A.dinv[i1]; }
        c.x[i0] = fma(alpha, q0, x0);
        const double s0 = fma(-alpha, m0, r0);
        const double z0 = jac ? s0 * d0 : s0;
        c.r[i0] = s0;
        acc[0] = fma(s0, z0, acc[0]); acc[1] = fma(s0, s0, acc[1]);
        if (h1) {
          c.x[i1] = fma(alpha, q1, x1);
          const double s1 = fma(-alpha, m1, r1);
          const double z1 = jac ? s1 * d1 : s1;
          c.r[i1] = s1;
          acc[0] = fma(s1, z1, acc[0]); acc[1] = fma(s1, s1, acc[1]);
        }
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
        const double ti = c.b[i] - spmv_row<OP_FP64>(c.A, c.x, i, c.x[i]);
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
