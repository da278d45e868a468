// cuth_fixed32.cuh -- ABLATION: the paper's fixed-FP32 PCG ("Fixed-Precision SpMV: standard FP64 and FP32
// kernels implemented directly via Algorithm 2"; Table VI: the fixed-FP32 column drifts to
// ||e||_inf = 0.64 K at the same iteration count).  Everything is single precision: the matrix is A2 (all four
// diagonals rounded to fp32, standard form, Alg. 2 as printed), x, r, p, mu are fp32 vectors, alpha / beta and the
// three dot products are fp32; the loop stops on ITS OWN recursive residual (Alg. 1 line 5) and never looks at
// b - A x -- which is exactly why it drifts.  SURVEY.md §8(f) rank 3; selected with CUTH_FIXED32.
//
// Not a performance path: one persistent cooperative kernel with the flat traversal (phases A / B / C separated by
// grid-wide barriers, as cuth_persistent.cuh), fixed-order fp32 reductions (bit-reproducible).  On exit x is widened
// into the caller's fp64 buffer and the TRUE fp64 residual b - A1 x is evaluated once, for the report only.
#pragma once
#include <cooperative_groups.h>

#include "cuth_persistent.cuh"

namespace cuth {

__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sums NV per-thread fp32 values over the whole grid in fp32, in a fixed order; result in all threads of all CTAs.
template <int NV>
__device__ __forceinline__ void grid_allreduce_f(cg::grid_group& grid, float (&v)[NV], float* partials, int& parity,
                                                 float* smem /* >= NV*32 + NV */) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = warp_sum_f(v[k]);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < NV; ++k) smem[k * 32 + wid] = v[k];
  __syncthreads();
  float* mine = partials + (size_t)parity * 3 * kPersistMaxBlocks;
  if (wid == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      const float t = warp_sum_f(lane < nw ? smem[k * 32 + lane] : 0.f);
      if (lane == 0) __stcg(&mine[k * kPersistMaxBlocks + blockIdx.x], t);
    }
  }
  grid.sync();
  if (wid < NV) {
    float a = 0.f;
    for (int b = lane; b < (int)gridDim.x; b += 32) a += __ldcg(&mine[wid * kPersistMaxBlocks + b]);
    a = warp_sum_f(a);
    if (lane == 0) smem[NV * 32 + wid] = a;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = smem[NV * 32 + k];
  __syncthreads();
  parity ^= 1;
}

// Row i of y = A2 v, Alg. 2 in fp32: entries of the fp32 copy, fp32 vector, fp32 fma.
__device__ __forceinline__ float spmv_row_f32(const DiaDev& A, const float* __restrict__ v, int64_t i, float vi) {
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  float acc = A.f0[i] * vi;
  if (i + 1 < n) acc = fmaf(A.f1[i], v[i + 1], acc);
  if (i >= 1) acc = fmaf(A.f1[i - 1], v[i - 1], acc);
  if (i + nx < n) acc = fmaf(A.f2[i], v[i + nx], acc);
  if (i >= nx) acc = fmaf(A.f2[i - nx], v[i - nx], acc);
  if (i + np < n) acc = fmaf(A.f3[i], v[i + np], acc);
  if (i >= np) acc = fmaf(A.f3[i - np], v[i - np], acc);
  return acc;
}

__global__ void __launch_bounds__(kPersistMaxThreads, 1) k_pcg_fixed32(const Ctx* __restrict__ ctxp, Ctl* ctl_g, double* partials_d) {
  cg::grid_group grid = cg::this_grid();
  __shared__ float smem[3 * 32 + 3];
  __shared__ double dsm[3 * 32 + 3];
  const Ctx c = *ctxp;
  const int64_t n = c.A.n;
  const int64_t gstride = (int64_t)gridDim.x * blockDim.x;
  const bool jac = c.jacobi != 0;
  float* partials = reinterpret_cast<float*>(partials_d);
  // fp32 vectors live in the fp64 workspace buffers (half of each is used)
  float* __restrict__ rf = reinterpret_cast<float*>(c.r);
  float* __restrict__ pf = reinterpret_cast<float*>(c.p);
  float* __restrict__ xf = reinterpret_cast<float*>(c.p2);
  float* __restrict__ mf = reinterpret_cast<float*>(c.mu);
  int parity = 0;
  int status = CUTH_SOLVE_RUNNING, it = 0;
  const bool refused = c.A.hdr[kHdrMagic] != kMagic;

  // ---- Alg. 1 lines 1-3 in fp32: x0, b rounded to fp32; r0 = b - A2 x0; z0 = r0 / D0; p0 = z0
  CUTH_ROWS(i) xf[i] = (float)c.x[i];
  grid.sync();
  float acc3[3] = {0.f, 0.f, 0.f};
  CUTH_ROWS(i) {
    const float bi = (float)c.b[i];
    const float ri = bi - spmv_row_f32(c.A, xf, i, xf[i]);
    const float zi = jac ? ri / c.A.f0[i] : ri;
    rf[i] = ri; pf[i] = zi;
    acc3[0] = fmaf(ri, zi, acc3[0]); acc3[1] = fmaf(ri, ri, acc3[1]); acc3[2] = fmaf(bi, bi, acc3[2]);
  }
  grid_allreduce_f<3>(grid, acc3, partials, parity, smem);
  float rho = acc3[0], rr = acc3[1];
  const float bb = acc3[2];
  const float tol2 = (float)c.rtol * (float)c.rtol * bb;
  if (refused) status = CUTH_SOLVE_BAD_MATRIX;
  else if (bb == 0.f) status = CUTH_SOLVE_CONVERGED;
  else if (rr <= tol2) status = CUTH_SOLVE_CONVERGED_UNVERIFIED;

  while (status == CUTH_SOLVE_RUNNING) {                        // Alg. 1 line 5
    float a1[1] = {0.f};
    CUTH_ROWS(i) {                                              // line 6
      const float pi = pf[i];
      const float m = spmv_row_f32(c.A, pf, i, pi);
      mf[i] = m;
      a1[0] = fmaf(pi, m, a1[0]);
    }
    grid_allreduce_f<1>(grid, a1, partials, parity, smem);
    const float pAp = a1[0];
    if (!(pAp > 0.f) || !(pAp <= 3.0e38f)) { status = CUTH_SOLVE_BREAKDOWN; break; }
    const float alpha = rho / pAp;                              // line 7
    float a2[2] = {0.f, 0.f};
    CUTH_ROWS(i) {
      xf[i] = fmaf(alpha, pf[i], xf[i]);                        // line 8
      const float ri = fmaf(-alpha, mf[i], rf[i]);              // line 9
      const float zi = jac ? ri / c.A.f0[i] : ri;               // line 10
      rf[i] = ri;
      a2[0] = fmaf(ri, zi, a2[0]); a2[1] = fmaf(ri, ri, a2[1]);
    }
    grid_allreduce_f<2>(grid, a2, partials, parity, smem);
    const float rho_new = a2[0];
    rr = a2[1];
    const float beta = rho_new / rho;                           // line 11
    rho = rho_new;
    ++it;                                                       // line 13
    if (!(rr == rr) || !(rho_new == rho_new)) { status = CUTH_SOLVE_BREAKDOWN; break; }
    if (rr <= tol2) { status = CUTH_SOLVE_CONVERGED_UNVERIFIED; break; }
    if (it >= c.max_iters) { status = CUTH_SOLVE_MAX_ITERS; break; }
    CUTH_ROWS(i) {                                              // line 12
      const float ri = rf[i];
      pf[i] = fmaf(beta, pf[i], jac ? ri / c.A.f0[i] : ri);
    }
    grid.sync();
  }

  // ---- report: x widened to fp64; true residual b - A1 x in fp64 (never used by the loop)
  if (!refused) {
    if (bb == 0.f) { CUTH_ROWS(i) c.x[i] = 0.0; }
    else { CUTH_ROWS(i) c.x[i] = (double)xf[i]; }
  }
  grid.sync();
  double t2[2] = {0.0, 0.0};
  if (!refused) {
    CUTH_ROWS(i) {
      const double bi = c.b[i];
      const double ti = bi - spmv_row<OP_FP64>(c.A, c.x, i, c.x[i]);
      t2[0] = fma(ti, ti, t2[0]); t2[1] = fma(bi, bi, t2[1]);
    }
  }
  int dparity = 0;
  grid_allreduce<2>(grid, t2, partials_d + 4 * kMaxBlocks - 2 * 3 * kPersistMaxBlocks, dparity, dsm);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    cuth_result_t res;
    res.status = status;
    res.iterations = it;
    res.promotions = 0; res.true_resid_evals = 1;
    res.rel_resid_true = t2[1] > 0.0 ? sqrt(t2[0] / t2[1]) : 0.0;
    res.rel_resid_rec = bb > 0.f ? (double)sqrtf(rr / bb) : 0.0;
    res.switch_reason = 0; res.switch_iteration = 0; res.switch_mask = 0;
    res.hard_restarts = 0; res.soft_restarts = 0; res.reserved = 0;
    *c.result = res;
  }
}

}  // namespace cuth
