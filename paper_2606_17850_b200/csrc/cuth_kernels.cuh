// cuth_kernels.cuh -- the PCG hot-path kernels (steps a1-a6 of DESIGN.md §3).
// Alg. 1 with M = diag(A); Alg. 2 for the SpMV.
#pragma once
#include "cuth_internal.cuh"
#include "cuth_policy.cuh"

namespace cuth {

constexpr int kThreads = 256;
constexpr int kRows = 2;        // rows per thread per tile (strided by blockDim for coalescing)

// ---------------------------------------------------------------------------------------------
// One row of y = A v, Alg. 2 read 0-based: 7 terms, out-of-range terms dropped.  The structural
// zeros stored in D1/D2 (x = nx-1, y = ny-1) make the lateral wrap-around vanish by themselves,
// so the operator is purely banded in the linear index i.
// OP = 0: fp64 matrix A1 (kernel K1 of the paper).
// OP = 1: fp32-stored off-diagonals promoted to fp64 (K3) and applied in
//         difference form  y_i = s_i v_i + sum_j g_ij (v_i - v_j)   (DESIGN.md R-F3).
// OP = 2: ABLATION (CUTH_MIXED_STD32): the paper's K3 literally -- all four diagonals of the fp32-rounded copy A2,
//         D0 included, promoted to fp64 and applied in standard form.
constexpr int OP_FP64 = 0, OP_DIFF32 = 1, OP_STD32 = 2;
template <int OP>
__device__ __forceinline__ double spmv_row(const DiaDev& A, const double* __restrict__ v, int64_t i, double vi) {
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = i + np < n, lo3 = i >= np;
  if (OP == OP_STD32) {
    const double a0 = (double)A.f0[i];
    const double a1u = up1 ? (double)A.f1[i] : 0.0, a1l = lo1 ? (double)A.f1[i - 1] : 0.0;
    const double a2u = up2 ? (double)A.f2[i] : 0.0, a2l = lo2 ? (double)A.f2[i - nx] : 0.0;
    const double a3u = up3 ? (double)A.f3[i] : 0.0, a3l = lo3 ? (double)A.f3[i - np] : 0.0;
    const double v1u = up1 ? v[i + 1] : 0.0, v1l = lo1 ? v[i - 1] : 0.0;
    const double v2u = up2 ? v[i + nx] : 0.0, v2l = lo2 ? v[i - nx] : 0.0;
    const double v3u = up3 ? v[i + np] : 0.0, v3l = lo3 ? v[i - np] : 0.0;
    double acc = a0 * vi;
    acc = fma(a1u, v1u, acc); acc = fma(a1l, v1l, acc);
    acc = fma(a2u, v2u, acc); acc = fma(a2l, v2l, acc);
    acc = fma(a3u, v3u, acc); acc = fma(a3l, v3l, acc);
    return acc;
  } else if (OP == OP_FP64) {
    // issue all loads first
    const double a0 = A.d0[i];
    const double a1u = up1 ? A.d1[i] : 0.0, a1l = lo1 ? A.d1[i - 1] : 0.0;
    const double a2u = up2 ? A.d2[i] : 0.0, a2l = lo2 ? A.d2[i - nx] : 0.0;
    const double a3u = up3 ? A.d3[i] : 0.0, a3l = lo3 ? A.d3[i - np] : 0.0;
    const double v1u = up1 ? v[i + 1] : 0.0, v1l = lo1 ? v[i - 1] : 0.0;
    const double v2u = up2 ? v[i + nx] : 0.0, v2l = lo2 ? v[i - nx] : 0.0;
    const double v3u = up3 ? v[i + np] : 0.0, v3l = lo3 ? v[i - np] : 0.0;
    double acc = a0 * vi;
    acc = fma(a1u, v1u, acc); acc = fma(a1l, v1l, acc);
    acc = fma(a2u, v2u, acc); acc = fma(a2l, v2l, acc);
    acc = fma(a3u, v3u, acc); acc = fma(a3l, v3l, acc);
    return acc;
  } else {
    const float g1u = up1 ? A.f1[i] : 0.f, g1l = lo1 ? A.f1[i - 1] : 0.f;
    const float g2u = up2 ? A.f2[i] : 0.f, g2l = lo2 ? A.f2[i - nx] : 0.f;
    const float g3u = up3 ? A.f3[i] : 0.f, g3l = lo3 ? A.f3[i - np] : 0.f;
    const double v1u = up1 ? v[i + 1] : vi, v1l = lo1 ? v[i - 1] : vi;
    const double v2u = up2 ? v[i + nx] : vi, v2l = lo2 ? v[i - nx] : vi;
    const double v3u = up3 ? v[i + np] : vi, v3l = lo3 ? v[i - np] : vi;
    const unsigned z = (unsigned)i / (unsigned)np;
    double acc = A.s_layer[z] * vi;
    // stored entries are A's (negative); conductance g = -entry, y += g (vi - vj) = entry (vj - vi)
    acc = fma((double)g1u, v1u - vi, acc); acc = fma((double)g1l, v1l - vi, acc);
    acc = fma((double)g2u, v2u - vi, acc); acc = fma((double)g2l, v2l - vi, acc);
    acc = fma((double)g3u, v3u - vi, acc); acc = fma((double)g3l, v3l - vi, acc);
    return acc;
  }
}

#define CUTH_TILE_LOOP(n_)                                                                   \
  for (int64_t base = (int64_t)blockIdx.x * (kThreads * kRows); base < (n_);                 \
       base += (int64_t)gridDim.x * (kThreads * kRows))

// ---------------------------------------------------------------------------------------------
// z-marching form of the same operator for grids whose x-y plane is too large for the +-nx*ny
// neighbours to survive in L2 (cfg 3, cfg 4): a CTA owns a ZTX x ZTY tile of the plane, each thread
// owns one (x, y) column and walks z = 0..nz-1 keeping v[z-1], v[z], v[z+1] and D3[z-1] in
// registers, so every matrix element and every vector element is fetched from HBM exactly once;
// the in-plane neighbours (+-1, +-nx) come through L1/L2.
#ifndef CUTH_ZTX
#define CUTH_ZTX 64
#endif
#ifndef CUTH_MINB
#define CUTH_MINB 4
#endif
constexpr int ZTX = CUTH_ZTX, ZTY = kThreads / CUTH_ZTX;   // ZTX * ZTY == kThreads
static_assert(ZTX * ZTY == kThreads, "tile must match the block size");

template <bool MIXED, class F>
__device__ __forceinline__ void zmarch_apply(const DiaDev& A, const double* __restrict__ v, F&& f) {
  const int tx = threadIdx.x % ZTX, ty = threadIdx.x / ZTX;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + ZTX - 1) / ZTX, tiles_y = (nyi + ZTY - 1) / ZTY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x = bx * ZTX + tx, y = by * ZTY + ty;
    if (x >= nxi || y >= nyi) continue;
    const int64_t c = x + nx * (int64_t)y;
    double v_lo = 0.0, v_c = v[c];
    double a3l = 0.0;     // D3[i - np] (fp64) or its fp32 value promoted
#pragma unroll 2
    for (int z = 0; z < nz; ++z) {
      const int64_t i = c + (int64_t)z * np;
      const bool up3 = z + 1 < nz, lo3 = z > 0;
      const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx;
      double acc, a3u, v_hi;
      if (!MIXED) {
        const double a0 = A.d0[i];
        const double a1u = up1 ? A.d1[i] : 0.0, a1l = lo1 ? A.d1[i - 1] : 0.0;
        const double a2u = up2 ? A.d2[i] : 0.0, a2l = lo2 ? A.d2[i - nx] : 0.0;
        a3u = up3 ? A.d3[i] : 0.0;
        v_hi = up3 ? v[i + np] : 0.0;
        const double v1u = up1 ? v[i + 1] : 0.0, v1l = lo1 ? v[i - 1] : 0.0;
        const double v2u = up2 ? v[i + nx] : 0.0, v2l = lo2 ? v[i - nx] : 0.0;
        acc = a0 * v_c;
        acc = fma(a1u, v1u, acc); acc = fma(a1l, v1l, acc);
        acc = fma(a2u, v2u, acc); acc = fma(a2l, v2l, acc);
        acc = fma(a3u, v_hi, acc); acc = fma(a3l, v_lo, acc);
      } else {
        const float g1u = up1 ? A.f1[i] : 0.f, g1l = lo1 ? A.f1[i - 1] : 0.f;
        const float g2u = up2 ? A.f2[i] : 0.f, g2l = lo2 ? A.f2[i - nx] : 0.f;
        a3u = up3 ? (double)A.f3[i] : 0.0;
        v_hi = up3 ? v[i + np] : v_c;
        const double v1u = up1 ? v[i + 1] : v_c, v1l = lo1 ? v[i - 1] : v_c;
        const double v2u = up2 ? v[i + nx] : v_c, v2l = lo2 ? v[i - nx] : v_c;
        acc = A.s_layer[z] * v_c;
        acc = fma((double)g1u, v1u - v_c, acc); acc = fma((double)g1l, v1l - v_c, acc);
        acc = fma((double)g2u, v2u - v_c, acc); acc = fma((double)g2l, v2l - v_c, acc);
        acc = fma(a3u, v_hi - v_c, acc);
        acc = fma(a3l, (lo3 ? v_lo : v_c) - v_c, acc);
      }
      f(i, v_c, acc);
      v_lo = v_c; v_c = v_hi; a3l = a3u;
    }
  }
}

// The same traversal with two x-adjacent columns per thread (nx even: every row starts at an even index, so
// v, D0 and D1 pairs are aligned 16-byte loads; D2 / D3 start at odd elements of the packed buffer, R-G5b,
// and stay scalar; the fp32 copy likewise).  Halves the index / predicate instructions per row, which is
// what bounds the one-column version (ncu: ~100 instructions per row, issue slots ~50 % busy).
template <bool MIXED, class F>
__device__ __forceinline__ void zmarch_apply_x2(const DiaDev& A, const double* __restrict__ v, F&& f) {
  const int tx = threadIdx.x % ZTX, ty = threadIdx.x / ZTX;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + 2 * ZTX - 1) / (2 * ZTX), tiles_y = (nyi + ZTY - 1) / ZTY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  auto ld2 = [](const double* p) { return *reinterpret_cast<const double2*>(p); };
  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x = bx * 2 * ZTX + 2 * tx, y = by * ZTY + ty;
    if (x >= nxi || y >= nyi) continue;
    const int64_t c0 = x + nx * (int64_t)y;
    double2 v_lo = make_double2(0.0, 0.0), v_c = ld2(v + c0);
    double a3l0 = 0.0, a3l1 = 0.0;
#pragma unroll 2
    for (int z = 0; z < nz; ++z) {
      const int64_t i = c0 + (int64_t)z * np;
      const bool up3 = z + 1 < nz, up2 = i + nx < n, lo2 = i >= nx, lo1 = i >= 1, up1 = i + 2 < n;
      double a1a, a1b = 0.0, a1l, a2u0 = 0.0, a2u1 = 0.0, a2l0 = 0.0, a2l1 = 0.0, a3u0 = 0.0, a3u1 = 0.0;
      double2 d0 = make_double2(0.0, 0.0);
      if (!MIXED) {
        d0 = ld2(A.d0 + i);
        if (up1) { const double2 d1 = ld2(A.d1 + i); a1a = d1.x; a1b = d1.y; } else { a1a = A.d1[i]; }
        a1l = lo1 ? A.d1[i - 1] : 0.0;
        if (up2) { a2u0 = A.d2[i]; a2u1 = A.d2[i + 1]; }
        if (lo2) { a2l0 = A.d2[i - nx]; a2l1 = A.d2[i + 1 - nx]; }
        if (up3) { a3u0 = A.d3[i]; a3u1 = A.d3[i + 1]; }
      } else {
        if (up1) { const float2 g = *reinterpret_cast<const float2*>(A.f1 + i); a1a = (double)g.x; a1b = (double)g.y; }
        else { a1a = (double)A.f1[i]; }
        a1l = lo1 ? (double)A.f1[i - 1] : 0.0;
        if (up2) { const float2 g = *reinterpret_cast<const float2*>(A.f2 + i); a2u0 = (double)g.x; a2u1 = (double)g.y; }
        if (lo2) { const float2 g = *reinterpret_cast<const float2*>(A.f2 + i - nx); a2l0 = (double)g.x; a2l1 = (double)g.y; }
        if (up3) { const float2 g = *reinterpret_cast<const float2*>(A.f3 + i); a3u0 = (double)g.x; a3u1 = (double)g.y; }
      }
      // absent neighbours: their matrix entry is 0 (standard form) / they take the centre value (difference form)
      const double2 zero2 = make_double2(0.0, 0.0);
      const double2 v_hi = up3 ? ld2(v + i + np) : (MIXED ? v_c : zero2);
      const double2 v2u = up2 ? ld2(v + i + nx) : (MIXED ? v_c : zero2);
      const double2 v2l = lo2 ? ld2(v + i - nx) : (MIXED ? v_c : zero2);
      const double vl = lo1 ? v[i - 1] : (MIXED ? v_c.x : 0.0), vr = up1 ? v[i + 2] : (MIXED ? v_c.y : 0.0);
      double y0, y1;
      if (!MIXED) {
        y0 = d0.x * v_c.x;              y1 = d0.y * v_c.y;
        y0 = fma(a1a, v_c.y, y0);       y1 = fma(a1a, v_c.x, y1);
        y0 = fma(a1l, vl, y0);          y1 = fma(a1b, vr, y1);
        y0 = fma(a2u0, v2u.x, y0);      y1 = fma(a2u1, v2u.y, y1);
        y0 = fma(a2l0, v2l.x, y0);      y1 = fma(a2l1, v2l.y, y1);
        y0 = fma(a3u0, v_hi.x, y0);     y1 = fma(a3u1, v_hi.y, y1);
        y0 = fma(a3l0, v_lo.x, y0);     y1 = fma(a3l1, v_lo.y, y1);
      } else {
        const double s = A.s_layer[z];
        const double2 lo = z > 0 ? v_lo : v_c;
        y0 = s * v_c.x;                         y1 = s * v_c.y;
        y0 = fma(a1a, v_c.y - v_c.x, y0);       y1 = fma(a1a, v_c.x - v_c.y, y1);
        y0 = fma(a1l, vl - v_c.x, y0);          y1 = fma(a1b, vr - v_c.y, y1);
        y0 = fma(a2u0, v2u.x - v_c.x, y0);      y1 = fma(a2u1, v2u.y - v_c.y, y1);
        y0 = fma(a2l0, v2l.x - v_c.x, y0);      y1 = fma(a2l1, v2l.y - v_c.y, y1);
        y0 = fma(a3u0, v_hi.x - v_c.x, y0);     y1 = fma(a3u1, v_hi.y - v_c.y, y1);
        y0 = fma(a3l0, lo.x - v_c.x, y0);       y1 = fma(a3l1, lo.y - v_c.y, y1);
      }
      f(i, v_c.x, y0);
      f(i + 1, v_c.y, y1);
      v_lo = v_c; v_c = v_hi; a3l0 = a3u0; a3l1 = a3u1;
    }
  }
}

// y_i = (A v)_i handed to f(i, v_i, y_i) for every row, with the traversal chosen at build time.
template <int OP, class F>
__device__ __forceinline__ void apply_A(const DiaDev& A, const double* __restrict__ v, F&& f) {
  constexpr bool MIXED = OP == OP_DIFF32;
  if (OP != OP_STD32 && A.zmarch) {              // the ablation operator exists in the flat traversal only
    if (A.x2) zmarch_apply_x2<MIXED>(A, v, f);
    else zmarch_apply<MIXED>(A, v, f);
  } else {
    CUTH_TILE_LOOP(A.n) {
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * kThreads;
        if (i < A.n) {
          const double vi = v[i];
          f(i, vi, spmv_row<OP>(A, v, i, vi));
        }
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Standalone SpMV (cuth_spmv).
template <int OP>
__global__ void __launch_bounds__(kThreads, CUTH_MINB) k_spmv_only(DiaDev A, const double* __restrict__ x, double* __restrict__ y) {
  apply_A<OP>(A, x, [&](int64_t i, double, double yi) { y[i] = yi; });
}

// Writes the per-call context and clears the control block (plain launch before the graph).
__global__ void k_set_ctx(Ctx c, Ctx* dst, Ctl* ctl) {
  if (threadIdx.x == 0) {
    *dst = c;
    Ctl z;
    memset(&z, 0, sizeof(z));
    z.status = CUTH_SOLVE_RUNNING;
    *ctl = z;
  }
}

// The same for a batch served by one cluster per right-hand side: context s = the base context with b, x, result moved to
// right-hand side s (vectors are right-hand-side-major, [nrhs][n]).
__global__ void k_set_ctx_batch(Ctx c, Ctx* dst, Ctl* ctl, int nrhs) {
  const int s = threadIdx.x;
  if (s < nrhs) {
    Ctx m = c;
    m.b = c.b + (size_t)s * (size_t)c.A.n;
    m.x = c.x + (size_t)s * (size_t)c.A.n;
    m.result = c.result + s;
    dst[s] = m;
    Ctl z;
    memset(&z, 0, sizeof(z));
    z.status = CUTH_SOLVE_RUNNING;
    ctl[s] = z;
  }
}

// rhs of eq. (5), T_amb = 0:  b = P + (C V / dt) T_n
__global__ void __launch_bounds__(kThreads) k_transient_rhs(DiaDev A, const double* __restrict__ power,
                                                           const double* __restrict__ t_n, double* __restrict__ b) {
  CUTH_TILE_LOOP(A.n) {
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      const int64_t i = base + threadIdx.x + k * kThreads;
      if (i < A.n) {
        const unsigned z = (unsigned)i / (unsigned)A.nxny;
        b[i] = __dadd_rn(power[i], __dmul_rn(A.cap_layer[z], t_n[i]));
      }
    }
  }
}

// Alg. 1 lines 1-3: r0 = b - A1 x0, z0 = M^-1 r0, rho = r.z, ||r||^2, ||b||^2; p := 0, beta := 0
// (the first k_pupdate then gives p0 = z0).
__global__ void __launch_bounds__(kThreads) k_init(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials,
                                                  cudaGraphConditionalHandle h_while) {
  __shared__ double smem[3 * 32];
  __shared__ int s_flag;
  const Ctx c = *ctxp;
  double acc[3] = {0.0, 0.0, 0.0};
  apply_A<OP_FP64>(c.A, c.x, [&](int64_t i, double, double ax) {
    const double bi = c.b[i];
    const double ri = bi - ax;
    const double zi = c.jacobi ? ri * c.A.dinv[i] : ri;
    c.r[i] = ri;
    c.p[i] = 0.0;
    acc[0] = fma(ri, zi, acc[0]);
    acc[1] = fma(ri, ri, acc[1]);
    acc[2] = fma(bi, bi, acc[2]);
  });
  if (grid_sum_last_block<3>(acc, partials, &ctl->ticket[0], smem, &s_flag) && threadIdx.x == 0) {
    const unsigned go = policy_init(ctl, c, acc[0], acc[1], acc[2]);
    cudaGraphSetConditional(h_while, go);
  }
}

// Alg. 1 line 12 (with line 10 recomputed): p = M^-1 r + beta p.
__global__ void __launch_bounds__(kThreads) k_pupdate(const Ctx* __restrict__ ctxp, const Ctl* __restrict__ ctl) {
  const Ctx c = *ctxp;
  const double beta = ctl->beta;
  const double* __restrict__ zs = c.cheb ? c.cz : c.r;     // Chebyshev: z = q(A) r is a stored vector
  CUTH_TILE_LOOP(c.A.n) {
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      const int64_t i = base + threadIdx.x + k * kThreads;
      if (i < c.A.n) {
        const double ri = zs[i];
        const double zi = c.jacobi ? ri * c.A.dinv[i] : ri;
        c.p[i] = fma(beta, c.p[i], zi);
      }
    }
  }
}

// Alg. 1 line 6 + the p.mu half of line 7: mu = A p (stage-dependent operator), pAp = p.mu.
template <int OP>
__device__ __forceinline__ void spmv_dot_body(const Ctx& c, double& acc) {
  apply_A<OP>(c.A, c.p, [&](int64_t i, double pi, double m) {
    c.mu[i] = m;
    acc = fma(pi, m, acc);
  });
}

__global__ void __launch_bounds__(kThreads, CUTH_MINB) k_spmv_dot(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials) {
  __shared__ double smem[32];
  __shared__ int s_flag;
  const Ctx c = *ctxp;
  double acc[1] = {0.0};
  if (ctl->stage != 0) spmv_dot_body<OP_FP64>(c, acc[0]);
  else if (c.early_op == OP_STD32) spmv_dot_body<OP_STD32>(c, acc[0]);
  else spmv_dot_body<OP_DIFF32>(c, acc[0]);
  if (grid_sum_last_block<1>(acc, partials, &ctl->ticket[1], smem, &s_flag) && threadIdx.x == 0) {
    policy_after_spmv(ctl, acc[0], false);      // Alg. 1 line 7
  }
}

// Alg. 1 lines 8-11: x += alpha p, r -= alpha mu, z = M^-1 r, rho' = r.z, ||r||^2; the last block
// forms beta, advances the iteration counter and takes the loop / policy decisions.
template <bool UPDATE_X>
__global__ void __launch_bounds__(1024) k_update(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials,
                                                    cudaGraphConditionalHandle h_while,
                                                    cudaGraphConditionalHandle h_if) {
  __shared__ double smem[2 * 32];
  __shared__ int s_flag;
  if (ctl->halt) return;                     // unrolled graph body: this pass is over (cuth_api.cu build_graph)
  const Ctx c = *ctxp;
  const double alpha = ctl->alpha;
  const int nt = (int)blockDim.x;            // threads per CTA are a launch parameter (k2_threads, cuth_api.cu)
  double acc[2] = {0.0, 0.0};
  if (!UPDATE_X && ctl->xnow) {
    // Fused path, an evaluation of the true residual is certain to follow this iteration (policy_after_spmv): Alg. 1
    // line 8 here instead of in the next K1 -- p' is the buffer K1 has just written (most of it still in L2).
    const double* __restrict__ pn = ctl->pcur ? c.p2 : c.p;
    for (int64_t base = (int64_t)blockIdx.x * (nt * kRows); base < c.A.n; base += (int64_t)gridDim.x * (nt * kRows)) {
      double xv[kRows], pv[kRows];
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * nt;
        xv[k] = i < c.A.n ? c.x[i] : 0.0; pv[k] = i < c.A.n ? pn[i] : 0.0;
      }
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * nt;
        if (i < c.A.n) c.x[i] = fma(alpha, pv[k], xv[k]);
      }
    }
  }
  if (!UPDATE_X && (c.A.n & 1) == 0) {
    // K2 of the fused path (32 B/row, nothing but streaming): rows in pairs as 16-byte accesses, two pairs per thread
    // per trip with all six loads issued before the first store -- 96 bytes in flight per thread instead of 48.
    const int64_t n2 = c.A.n >> 1;
    const double2* __restrict__ r2 = reinterpret_cast<const double2*>(c.r);
    const double2* __restrict__ m2 = reinterpret_cast<const double2*>(c.mu);
    const double2* __restrict__ d2 = reinterpret_cast<const double2*>(c.A.dinv);
    // early stage of the fused path: M^-1 = fp32(1/D0), the same values K1 forms z = M^-1 r with (cuth_fused*.cuh)
    const float2* __restrict__ f2 = reinterpret_cast<const float2*>(c.A.dinv32);
    const bool m32 = ctl->stage == 0;
    double2* __restrict__ w2 = reinterpret_cast<double2*>(c.r);
    const bool jac = c.jacobi != 0;
#ifndef CUTH_K2_PAIRS
#define CUTH_K2_PAIRS 2
#endif
    constexpr int NP = CUTH_K2_PAIRS;
    for (int64_t base = (int64_t)blockIdx.x * (nt * NP); base < n2; base += (int64_t)gridDim.x * (nt * NP)) {
      const double2 one = make_double2(1.0, 1.0), zero = make_double2(0.0, 0.0);
      double2 rv[NP], mv[NP], dv[NP];
      bool h[NP];
#pragma unroll
      for (int q = 0; q < NP; ++q) {
        const int64_t i = base + threadIdx.x + (int64_t)q * nt;
        h[q] = i < n2;
        rv[q] = h[q] ? r2[i] : zero;
        mv[q] = h[q] ? __ldcs(&m2[i]) : zero;
        dv[q] = one;
        if (jac && h[q]) {
          if (m32) { const float2 f = f2[i]; dv[q] = make_double2((double)f.x, (double)f.y); }
          else dv[q] = d2[i];
        }
      }
#pragma unroll
      for (int q = 0; q < NP; ++q) {
        const int64_t i = base + threadIdx.x + (int64_t)q * nt;
        const double a0 = fma(-alpha, mv[q].x, rv[q].x), a1 = fma(-alpha, mv[q].y, rv[q].y);
        if (h[q]) w2[i] = make_double2(a0, a1);
        acc[0] = fma(a0, a0 * dv[q].x, acc[0]); acc[1] = fma(a0, a0, acc[1]);
        acc[0] = fma(a1, a1 * dv[q].y, acc[0]); acc[1] = fma(a1, a1, acc[1]);
      }
    }
  } else {
  for (int64_t base = (int64_t)blockIdx.x * (nt * kRows); base < c.A.n; base += (int64_t)gridDim.x * (nt * kRows)) {
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      const int64_t i = base + threadIdx.x + k * nt;
      if (i < c.A.n) {
        if (UPDATE_X) c.x[i] = fma(alpha, c.p[i], c.x[i]);
        const double ri = fma(-alpha, c.mu[i], c.r[i]);
        const double zi = c.jacobi ? ri * ((!UPDATE_X && ctl->stage == 0) ? (double)c.A.dinv32[i] : c.A.dinv[i]) : ri;
        c.r[i] = ri;
        acc[0] = fma(ri, zi, acc[0]);
        acc[1] = fma(ri, ri, acc[1]);
      }
    }
  }
  }
  if (grid_sum_last_block<2>(acc, partials + kMaxBlocks, &ctl->ticket[2], smem, &s_flag) && threadIdx.x == 0) {
    unsigned go, want;
    policy_after_update(ctl, c, acc[0], acc[1], go, want);
    if (!ctl->no_graph) { cudaGraphSetConditional(h_while, go); cudaGraphSetConditional(h_if, want); }
  }
}

// True residual: t = b - A1 x in fp64, ||t||^2 and the drift ||t - r||^2; the last block applies the
// stopping rule and eq. (14a)-(14c).  t itself is not stored (round 2b wrote it to the mu buffer for k_restart: 8 of the
// 64 B/row of every evaluation for a restart that happens once or twice per solve): k_restart forms it again.
__global__ void __launch_bounds__(kThreads) k_true_resid(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials,
                                                        cudaGraphConditionalHandle h_while) {
  __shared__ double smem[2 * 32];
  __shared__ int s_flag;
  const Ctx c = *ctxp;
  double acc[2] = {0.0, 0.0};
  apply_A<OP_FP64>(c.A, c.x, [&](int64_t i, double, double ax) {
    const double ti = c.b[i] - ax;
    const double di = ti - c.r[i];
    acc[0] = fma(ti, ti, acc[0]);
    acc[1] = fma(di, di, acc[1]);
  });
  if (grid_sum_last_block<2>(acc, partials + 2 * kMaxBlocks, &ctl->ticket[3], smem, &s_flag) && threadIdx.x == 0) {
    const unsigned go = policy_after_true(ctl, c, acc[0], acc[1]);
    if (!ctl->no_graph) cudaGraphSetConditional(h_while, go);
  }
}

// Hot restart: r := t = b - A1 x (the same operations on the same x as in k_true_resid: the same bits),
// z = M^-1 r, rho = r.z, beta := 0 so that the next k_pupdate gives p = z (p's defining equation, Alg. 1 line 3).
// No-op unless ctl->restart.
__global__ void __launch_bounds__(kThreads) k_restart(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials) {
  __shared__ double smem[2 * 32];
  __shared__ int s_flag;
  const int mode = ctl->restart;
  if (!mode) return;
  const Ctx c = *ctxp;
  double acc[2] = {0.0, 0.0};
  apply_A<OP_FP64>(c.A, c.x, [&](int64_t i, double, double ax) {
    const double ri = c.b[i] - ax;
    const double zi = c.jacobi ? ri * c.A.dinv[i] : ri;
    c.r[i] = ri;
    acc[0] = fma(ri, zi, acc[0]);
    acc[1] = fma(ri, ri, acc[1]);
  });
  if (grid_sum_last_block<2>(acc, partials + 2 * kMaxBlocks, &ctl->ticket[4], smem, &s_flag) && threadIdx.x == 0) {
    policy_after_restart(ctl, c, mode, acc[0], acc[1]);
  }
}

// Measurement hook support: marks the control block as "outside a graph"; early = 1 re-arms the early stage
// (fp32-stored operator) for the replayed kernels.
__global__ void k_mark_no_graph(Ctl* ctl, int early) {
  ctl->no_graph = 1; ctl->restart = 0; ctl->halt = 0;
  if (early) ctl->stage = 0;
}

// Writes the result record; x := 0 when b = 0.
__global__ void __launch_bounds__(kThreads) k_finalize(const Ctx* __restrict__ ctxp, Ctl* ctl) {
  const Ctx c = *ctxp;
  const double xalpha = ctl->xalpha;
  if (xalpha != 0.0 && !ctl->zero_rhs) {      // deferred x += alpha p of the last iteration (fused path)
    const double* p = ctl->pcur ? c.p2 : c.p;
    CUTH_TILE_LOOP(c.A.n) {
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * kThreads;
        if (i < c.A.n) c.x[i] = fma(xalpha, p[i], c.x[i]);
      }
    }
  }
  if (ctl->zero_rhs) {
    CUTH_TILE_LOOP(c.A.n) {
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * kThreads;
        if (i < c.A.n) c.x[i] = 0.0;
      }
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    write_result(ctl, c);
  }
}

}  // namespace cuth
