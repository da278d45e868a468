// cuth_batch.cuh -- several right-hand sides that share one matrix, solved in lock-step by ONE persistent
// cooperative kernel (SURVEY.md §8(f) "multi-RHS / batched solves sharing one A": the paper
// notes that direct solvers win when many right-hand sides share A; here the iterative path amortises A instead).
// Each right-hand side runs its own Alg. 1 recurrence -- own alpha, beta, rho, own stopping
// test and true-residual verification (cuth_policy.cuh, one Ctl per right-hand side) -- this is NOT block-CG:
// the iterates of right-hand side s are those a single solve would produce.  What is shared:
//   * every matrix row is fetched once per chunk of S right-hand sides and applied to S vectors;
//   * every grid-wide barrier and reduction serves all right-hand sides at once, so on the small grids where a
//     single solve is bound by the ~4.5 us per phase of the barrier the batch costs little more
//     than one solve.
// FP64 or MIXED (each right-hand side has its own stage and switches on its own, eq. (14a)-(14c)), M = diag(A) or I.
// Vectors are stored right-hand-side-major: v[s * n + i].
// Phases per iteration (as cuth_persistent.cuh): A  p = z + beta p | B  mu = A p, p.mu | C  x, r, r.z, ||r||^2 |
// D (on demand) t = b - A x | E (restart) r := t.  A right-hand side that has finished is skipped by every phase.
#pragma once
#include <cooperative_groups.h>

#include "cuth_kernels.cuh"

namespace cuth {

namespace cgb = cooperative_groups;

constexpr int kBatchMaxRhs = 32;
constexpr int kBatchChunk = 4;            // S: right-hand sides that share one fetch of a matrix row
constexpr int kBatchMaxBlocks = 1024;

struct BatchCtx {
  DiaDev A;
  const double* b; double* x; double* r; double* p; double* mu;   // [nrhs][n] each
  cuth_result_t* result;                                          // [nrhs]
  double rtol;
  int32_t nrhs, max_iters, jacobi, ntiles;   // ntiles: CTAs per chunk of S right-hand sides
  int32_t precision, period;                 // CUTH_FP64 / CUTH_MIXED; true-residual period of the MIXED early stage
};

struct BatchWorkspace {
  BatchCtx* ctx; Ctl* ctl; double* partials; double* r; double* p; double* mu;
  size_t bytes;
};

inline BatchWorkspace carve_batch_workspace(void* base, int64_t n, int nrhs) {
  BatchWorkspace w;
  char* c = (char*)base;
  size_t o = 0;
  w.ctx = (BatchCtx*)(c + o); o = align_up(o + sizeof(BatchCtx));
  w.ctl = (Ctl*)(c + o); o = align_up(o + sizeof(Ctl) * (size_t)kBatchMaxRhs);
  w.partials = (double*)(c + o); o = align_up(o + sizeof(double) * 2 * 3 * (size_t)kBatchMaxRhs * kBatchMaxBlocks);
  const size_t vec = sizeof(double) * (size_t)n * (size_t)nrhs;
  w.r = (double*)(c + o); o = align_up(o + vec);
  w.p = (double*)(c + o); o = align_up(o + vec);
  w.mu = (double*)(c + o); o = align_up(o + vec);
  w.bytes = o;
  return w;
}

#ifdef __CUDACC__

__global__ void k_batch_set_ctx(BatchCtx c, BatchCtx* dst, Ctl* ctl) {
  if (threadIdx.x == 0) *dst = c;
  if (threadIdx.x < kBatchMaxRhs) {
    Ctl z;
    memset(&z, 0, sizeof(z));
    z.status = CUTH_SOLVE_RUNNING;
    ctl[threadIdx.x] = z;
  }
}

// The seven coefficients of row i of A1 (Alg. 2; absent terms are 0) and their neighbour indices.
struct RowCoef {
  double a0, a1u, a1l, a2u, a2l, a3u, a3l;
  bool up1, lo1, up2, lo2, up3, lo3;
};

__device__ __forceinline__ RowCoef load_row(const DiaDev& A, int64_t i) {
  RowCoef q;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  q.up1 = i + 1 < n; q.lo1 = i >= 1; q.up2 = i + nx < n; q.lo2 = i >= nx; q.up3 = i + np < n; q.lo3 = i >= np;
  q.a0 = A.d0[i];
  q.a1u = q.up1 ? A.d1[i] : 0.0; q.a1l = q.lo1 ? A.d1[i - 1] : 0.0;
  q.a2u = q.up2 ? A.d2[i] : 0.0; q.a2l = q.lo2 ? A.d2[i - nx] : 0.0;
  q.a3u = q.up3 ? A.d3[i] : 0.0; q.a3l = q.lo3 ? A.d3[i - np] : 0.0;
  return q;
}

// Same order of operations as spmv_row<false>.
__device__ __forceinline__ double apply_row(const RowCoef& q, const DiaDev& A, const double* __restrict__ v, int64_t i,
                                            double vi) {
  const int64_t nx = A.nx, np = A.nxny;
  const double v1u = q.up1 ? v[i + 1] : 0.0, v1l = q.lo1 ? v[i - 1] : 0.0;
  const double v2u = q.up2 ? v[i + nx] : 0.0, v2l = q.lo2 ? v[i - nx] : 0.0;
  const double v3u = q.up3 ? v[i + np] : 0.0, v3l = q.lo3 ? v[i - np] : 0.0;
  double acc = q.a0 * vi;
  acc = fma(q.a1u, v1u, acc); acc = fma(q.a1l, v1l, acc);
  acc = fma(q.a2u, v2u, acc); acc = fma(q.a2l, v2l, acc);
  acc = fma(q.a3u, v3u, acc); acc = fma(q.a3l, v3l, acc);
  return acc;
}

// Row i of the fp32-stored operator (K3) applied in difference form (DESIGN.md R-F3); same loads and
// order of operations as spmv_row<true>.
struct RowCoef32 { float g1u, g1l, g2u, g2l, g3u, g3l; double s; };

__device__ __forceinline__ RowCoef32 load_row32(const DiaDev& A, const RowCoef& q, int64_t i) {
  RowCoef32 f;
  const int64_t nx = A.nx, np = A.nxny;
  f.g1u = q.up1 ? A.f1[i] : 0.f; f.g1l = q.lo1 ? A.f1[i - 1] : 0.f;
  f.g2u = q.up2 ? A.f2[i] : 0.f; f.g2l = q.lo2 ? A.f2[i - nx] : 0.f;
  f.g3u = q.up3 ? A.f3[i] : 0.f; f.g3l = q.lo3 ? A.f3[i - np] : 0.f;
  f.s = A.s_layer[(unsigned)i / (unsigned)np];
  return f;
}

__device__ __forceinline__ double apply_row32(const RowCoef32& f, const RowCoef& q, const DiaDev& A,
                                              const double* __restrict__ v, int64_t i, double vi) {
  const int64_t nx = A.nx, np = A.nxny;
  const double v1u = q.up1 ? v[i + 1] : vi, v1l = q.lo1 ? v[i - 1] : vi;
  const double v2u = q.up2 ? v[i + nx] : vi, v2l = q.lo2 ? v[i - nx] : vi;
  const double v3u = q.up3 ? v[i + np] : vi, v3l = q.lo3 ? v[i - np] : vi;
  double acc = f.s * vi;
  acc = fma((double)f.g1u, v1u - vi, acc); acc = fma((double)f.g1l, v1l - vi, acc);
  acc = fma((double)f.g2u, v2u - vi, acc); acc = fma((double)f.g2l, v2l - vi, acc);
  acc = fma((double)f.g3u, v3u - vi, acc); acc = fma((double)f.g3l, v3l - vi, acc);
  return acc;
}

// The index predicates of a row without its fp64 coefficients (early-stage-only chunks do not touch A1).
__device__ __forceinline__ RowCoef row_predicates(const DiaDev& A, int64_t i) {
  RowCoef q;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  q.up1 = i + 1 < n; q.lo1 = i >= 1; q.up2 = i + nx < n; q.lo2 = i >= nx; q.up3 = i + np < n; q.lo3 = i >= np;
  q.a0 = q.a1u = q.a1l = q.a2u = q.a2l = q.a3u = q.a3l = 0.0;
  return q;
}

// Block-level part of a batched reduction: NV values for each of the S right-hand sides of this CTA's chunk.
// partials layout: [parity][k * nrhs + s][kBatchMaxBlocks], indexed by the CTA's row-tile number.
template <int NV>
__device__ __forceinline__ void batch_deposit(double (&v)[NV * kBatchChunk], double* mine, int s0, int nrhs, int tile,
                                              double* smem) {
  block_sum<NV * kBatchChunk>(v, smem);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k)
#pragma unroll
      for (int s = 0; s < kBatchChunk; ++s)
        if (s0 + s < nrhs) __stcg(&mine[(size_t)(k * nrhs + s0 + s) * kBatchMaxBlocks + tile], v[k * kBatchChunk + s]);
  }
  __syncthreads();
}

// Grid-wide part: after the barrier every CTA adds the per-tile partials of all `count` = nv * nrhs values in the
// same fixed order, so all CTAs hold bitwise-identical sums in tot[] (shared memory) and take identical decisions.
__device__ __forceinline__ void batch_collect(cgb::grid_group& grid, const double* mine, int count, int ntiles,
                                              double* tot) {   // ntiles: tiles that own rows (the others deposit 0)
  grid.sync();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if (count <= nw) {            // at most one value per warp: keep the tile loop simple so that its loads overlap
    if (wid < count) {
      double a = 0.0;
#pragma unroll 4
      for (int b = lane; b < ntiles; b += 32) a += __ldcg(&mine[(size_t)wid * kBatchMaxBlocks + b]);
      a = warp_sum(a);
      if (lane == 0) tot[wid] = a;
    }
  } else {
    constexpr int U = 8;        // values a warp sums side by side: one L2 round trip for up to U * nw values
    for (int v0 = wid; v0 < count; v0 += U * nw) {
      double a[U];
#pragma unroll
      for (int u = 0; u < U; ++u) a[u] = 0.0;
      for (int b = lane; b < ntiles; b += 32) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const int v = v0 + u * nw;
          if (v < count) a[u] += __ldcg(&mine[(size_t)v * kBatchMaxBlocks + b]);
        }
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int v = v0 + u * nw;
        const double t = warp_sum(a[u]);
        if (lane == 0 && v < count) tot[v] = t;
      }
    }
  }
  __syncthreads();
}

// Rows of this CTA: row i = tile * kThreads + thread, then strides of ntiles * kThreads; identical in every phase,
// so only the stencil phases need a preceding grid-wide barrier.  One row at a time: the S right-hand sides of the
// chunk supply the independent loads.
#define CUTH_BROWS(i_)                                                                           \
  for (int64_t i_ = (int64_t)tile * kThreads + threadIdx.x; i_ < n; i_ += (int64_t)ntiles * kThreads)

// Grid: ntiles * ceil(nrhs / S) CTAs, all co-resident.  CTA (tile, chunk) owns the right-hand sides
// chunk*S .. chunk*S+S-1 on its rows; decisions for ALL right-hand sides are replicated in every CTA.
__global__ void __launch_bounds__(kThreads, 3) k_pcg_batch(const BatchCtx* __restrict__ ctxp, Ctl* ctl_g,
                                                          double* partials) {
  constexpr int S = kBatchChunk;
  cgb::grid_group grid = cgb::this_grid();
  __shared__ Ctl sc[kBatchMaxRhs];
  __shared__ double tot[3 * kBatchMaxRhs];
  __shared__ double smem[3 * S * 32];
  __shared__ int s_go[kBatchMaxRhs], s_want[kBatchMaxRhs], s_mode[kBatchMaxRhs], s_any[3];
  const BatchCtx c = *ctxp;
  const int64_t n = c.A.n;
  const int nrhs = c.nrhs, ntiles = c.ntiles;
  const int nact = (int)((n + kThreads - 1) / kThreads < (int64_t)ntiles ? (n + kThreads - 1) / kThreads : (int64_t)ntiles);
  const int tile = blockIdx.x % ntiles, s0 = (blockIdx.x / ntiles) * S;
  const bool jac = c.jacobi != 0;
  // the policy code reads its options from a Ctx: only these fields are consulted on this path
  Ctx pc;
  pc.A = c.A; pc.transient_call = 0;          // the matrix object's own header is checked by policy_init
  pc.rtol = c.rtol; pc.precision = c.precision; pc.max_iters = c.max_iters; pc.period = c.period; pc.cheb = 0;
  pc.soft_restart = 1; pc.soft_drift2 = 1e-2;       // as cuth_pcg_solve (DESIGN.md R-G11)
  int parity = 0;
  if (threadIdx.x < nrhs) sc[threadIdx.x] = ctl_g[threadIdx.x];      // cleared by k_batch_set_ctx
  __syncthreads();
  auto part = [&]() { return partials + (size_t)parity * 3 * kBatchMaxRhs * kBatchMaxBlocks; };
  size_t o[S];
#pragma unroll
  for (int s = 0; s < S; ++s) o[s] = (size_t)(s0 + s < nrhs ? s0 + s : 0) * (size_t)n;
  bool live[S];

  // ---- Alg. 1 lines 1-3
  {
    double acc[3 * S];
#pragma unroll
    for (int q = 0; q < 3 * S; ++q) acc[q] = 0.0;
    CUTH_BROWS(i) {
      const RowCoef rc = load_row(c.A, i);
      const double di = jac ? c.A.dinv[i] : 1.0;
      double bi[S], ri[S];
#pragma unroll
      for (int s = 0; s < S; ++s) {
        bi[s] = 0.0; ri[s] = 0.0;
        if (s0 + s < nrhs) {
          bi[s] = c.b[o[s] + i];
          ri[s] = bi[s] - apply_row(rc, c.A, c.x + o[s], i, c.x[o[s] + i]);
        }
      }
#pragma unroll
      for (int s = 0; s < S; ++s) {
        if (s0 + s < nrhs) {
          const double zi = ri[s] * di;
          c.r[o[s] + i] = ri[s];
          c.p[o[s] + i] = 0.0;
          acc[s] = fma(ri[s], zi, acc[s]); acc[S + s] = fma(ri[s], ri[s], acc[S + s]);
          acc[2 * S + s] = fma(bi[s], bi[s], acc[2 * S + s]);
        }
      }
    }
    batch_deposit<3>(acc, part(), s0, nrhs, tile, smem);
  }
  batch_collect(grid, part(), 3 * nrhs, nact, tot);
  parity ^= 1;
  if (threadIdx.x < nrhs) {
    const int s = threadIdx.x;
    s_go[s] = (int)policy_init(&sc[s], pc, tot[s], tot[nrhs + s], tot[2 * nrhs + s]);
    s_want[s] = 0; s_mode[s] = 0;
  }
  __syncthreads();
  if (threadIdx.x == 0) { int a = 0; for (int s = 0; s < nrhs; ++s) a |= s_go[s]; s_any[0] = a; }
  __syncthreads();

  while (s_any[0]) {
#pragma unroll
    for (int s = 0; s < S; ++s) live[s] = s0 + s < nrhs && s_go[s0 + s] != 0;
    // ---- A: p = z + beta p
    {
      double beta[S];
#pragma unroll
      for (int s = 0; s < S; ++s) beta[s] = live[s] ? sc[s0 + s].beta : 0.0;
      CUTH_BROWS(i) {
        const double di = jac ? c.A.dinv[i] : 1.0;
        double ri[S], pi[S];
#pragma unroll
        for (int s = 0; s < S; ++s) { ri[s] = live[s] ? c.r[o[s] + i] : 0.0; pi[s] = live[s] ? c.p[o[s] + i] : 0.0; }
#pragma unroll
        for (int s = 0; s < S; ++s)
          if (live[s]) c.p[o[s] + i] = fma(beta[s], pi[s], jac ? ri[s] * di : ri[s]);
      }
    }
    grid.sync();
    // ---- B: mu = A p, p.mu  (per right-hand side: the fp32-stored operator in its early stage, A1 after)
    {
      double acc[S];
      bool early[S];
      bool any_early = false, any_late = false;
#pragma unroll
      for (int s = 0; s < S; ++s) {
        acc[s] = 0.0;
        early[s] = live[s] && sc[s0 + s].stage == 0;
        any_early = any_early || early[s];
        any_late = any_late || (live[s] && !early[s]);
      }
      CUTH_BROWS(i) {
        const RowCoef rc = any_late ? load_row(c.A, i) : row_predicates(c.A, i);
        RowCoef32 rf;
        if (any_early) rf = load_row32(c.A, rc, i);
        double pi[S], m[S];
#pragma unroll
        for (int s = 0; s < S; ++s) {
          pi[s] = 0.0; m[s] = 0.0;
          if (live[s]) {
            pi[s] = c.p[o[s] + i];
            m[s] = early[s] ? apply_row32(rf, rc, c.A, c.p + o[s], i, pi[s]) : apply_row(rc, c.A, c.p + o[s], i, pi[s]);
          }
        }
#pragma unroll
        for (int s = 0; s < S; ++s)
          if (live[s]) { c.mu[o[s] + i] = m[s]; acc[s] = fma(pi[s], m[s], acc[s]); }
      }
      batch_deposit<1>(acc, part(), s0, nrhs, tile, smem);
    }
    batch_collect(grid, part(), nrhs, nact, tot);
    parity ^= 1;
    if (threadIdx.x < nrhs && s_go[threadIdx.x]) policy_after_spmv(&sc[threadIdx.x], tot[threadIdx.x], false);
    __syncthreads();
    // ---- C: x += alpha p, r -= alpha mu, r.z, ||r||^2
    {
      double alpha[S];
#pragma unroll
      for (int s = 0; s < S; ++s) alpha[s] = live[s] ? sc[s0 + s].alpha : 0.0;
      double acc[2 * S];
#pragma unroll
      for (int q = 0; q < 2 * S; ++q) acc[q] = 0.0;
      CUTH_BROWS(i) {
        const double di = jac ? c.A.dinv[i] : 1.0;
        double xi[S], pi[S], mi[S], ri[S];
#pragma unroll
        for (int s = 0; s < S; ++s) {
          xi[s] = pi[s] = mi[s] = ri[s] = 0.0;
          if (live[s]) { xi[s] = c.x[o[s] + i]; pi[s] = c.p[o[s] + i]; mi[s] = c.mu[o[s] + i]; ri[s] = c.r[o[s] + i]; }
        }
#pragma unroll
        for (int s = 0; s < S; ++s) {
          if (live[s]) {
            c.x[o[s] + i] = fma(alpha[s], pi[s], xi[s]);
            const double rn = fma(-alpha[s], mi[s], ri[s]);
            const double zi = jac ? rn * di : rn;
            c.r[o[s] + i] = rn;
            acc[s] = fma(rn, zi, acc[s]); acc[S + s] = fma(rn, rn, acc[S + s]);
          }
        }
      }
      batch_deposit<2>(acc, part(), s0, nrhs, tile, smem);
    }
    batch_collect(grid, part(), 2 * nrhs, nact, tot);
    parity ^= 1;
    if (threadIdx.x < nrhs && s_go[threadIdx.x]) {
      const int s = threadIdx.x;
      unsigned g_, w_;
      policy_after_update(&sc[s], pc, tot[s], tot[nrhs + s], g_, w_);
      s_go[s] = (int)g_; s_want[s] = (int)w_;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int a = 0, w = 0;
      for (int s = 0; s < nrhs; ++s) { a |= s_go[s]; w |= (s_go[s] && s_want[s]) ? 1 : 0; }
      s_any[0] = a; s_any[1] = w;
    }
    __syncthreads();
    if (s_any[1]) {
      // ---- D: true residual of the right-hand sides that asked for it (x is complete: the collect was a barrier)
#pragma unroll
      for (int s = 0; s < S; ++s) live[s] = s0 + s < nrhs && s_go[s0 + s] != 0 && s_want[s0 + s] != 0;
      {
        double acc[2 * S];
#pragma unroll
        for (int q = 0; q < 2 * S; ++q) acc[q] = 0.0;
        CUTH_BROWS(i) {
          const RowCoef rc = load_row(c.A, i);
          double ti[S], dd[S];
#pragma unroll
          for (int s = 0; s < S; ++s) {
            ti[s] = dd[s] = 0.0;
            if (live[s]) {
              ti[s] = c.b[o[s] + i] - apply_row(rc, c.A, c.x + o[s], i, c.x[o[s] + i]);
              dd[s] = ti[s] - c.r[o[s] + i];
            }
          }
#pragma unroll
          for (int s = 0; s < S; ++s)
            if (live[s]) { c.mu[o[s] + i] = ti[s]; acc[s] = fma(ti[s], ti[s], acc[s]); acc[S + s] = fma(dd[s], dd[s], acc[S + s]); }
        }
        batch_deposit<2>(acc, part(), s0, nrhs, tile, smem);
      }
      batch_collect(grid, part(), 2 * nrhs, nact, tot);
      parity ^= 1;
      if (threadIdx.x < nrhs) {
        const int s = threadIdx.x;
        s_mode[s] = 0;
        if (s_go[s] && s_want[s]) {
          s_go[s] = (int)policy_after_true(&sc[s], pc, tot[s], tot[nrhs + s]);
          s_mode[s] = s_go[s] ? sc[s].restart : 0;
        }
      }
      __syncthreads();
      if (threadIdx.x == 0) {
        int a = 0, m = 0;
        for (int s = 0; s < nrhs; ++s) { a |= s_go[s]; m |= s_mode[s]; }
        s_any[0] = a; s_any[2] = m;
      }
      __syncthreads();
      if (s_any[2]) {
        // ---- E: r := t for the right-hand sides whose verification failed
#pragma unroll
        for (int s = 0; s < S; ++s) live[s] = s0 + s < nrhs && s_mode[s0 + s] != 0;
        {
          double acc[2 * S];
#pragma unroll
          for (int q = 0; q < 2 * S; ++q) acc[q] = 0.0;
          CUTH_BROWS(i) {
            const double di = jac ? c.A.dinv[i] : 1.0;
#pragma unroll
            for (int s = 0; s < S; ++s) {
              if (live[s]) {
                const double ri = c.mu[o[s] + i];
                const double zi = jac ? ri * di : ri;
                c.r[o[s] + i] = ri;
                acc[s] = fma(ri, zi, acc[s]); acc[S + s] = fma(ri, ri, acc[S + s]);
              }
            }
          }
          batch_deposit<2>(acc, part(), s0, nrhs, tile, smem);
        }
        batch_collect(grid, part(), 2 * nrhs, nact, tot);
        parity ^= 1;
        if (threadIdx.x < nrhs && s_mode[threadIdx.x]) {
          const int s = threadIdx.x;
          policy_after_restart(&sc[s], pc, s_mode[s], tot[s], tot[nrhs + s]);
          s_mode[s] = 0;
        }
        __syncthreads();
      }
    }
  }
  // ---- epilogue
#pragma unroll
  for (int s = 0; s < S; ++s) {
    if (s0 + s < nrhs && sc[s0 + s].zero_rhs) { CUTH_BROWS(i) c.x[o[s] + i] = 0.0; }
  }
  if (blockIdx.x == 0 && threadIdx.x < nrhs) {
    const int s = threadIdx.x;
    sc[s].exiting = 0;
    pc.result = c.result + s;
    write_result(&sc[s], pc);
    ctl_g[s] = sc[s];
  }
}

#endif  // __CUDACC__

}  // namespace cuth
