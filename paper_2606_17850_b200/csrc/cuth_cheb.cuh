// cuth_cheb.cuh -- Chebyshev polynomial preconditioner (Alg. 3) and the Lanczos
// spectral-range estimate: SURVEY.md §8(f) rank 1, the paper's own preconditioner.
//
// One apply z = q(A) r of degree k is k-1 stencil kernels with NO reduction inside:
// with d and r_c eliminated in favour of the partial sums Z_j = d_0 + ... + d_{j-1} (see k_cheb_first below):
//   FIRST (i = 0)       Z_1 = r/theta formed on the fly (A Z_1 = (A r)/theta), Z_2
//   MID   (0 < i < k-2) Z_{i+2} = Z_{i+1} + c1[i] (Z_{i+1} - Z_i) + c2[i] (r - A Z_{i+1}), written over Z_i
//   LAST  (i = k-2)     z = Z_k (fp64), rho = r.z
// (Alg. 3's k-th SpMV and d-update feed nothing and are skipped: z is identical.)
// Element type T of d, rc, z: double (FP64 mode, fp64 matrix A1) or float (MIXED mode: "FP32 for all
// vector and scalar operations" of Alg. 3, on the fp32-stored matrix A2 in difference form).
#pragma once
#include "cuth_kernels.cuh"

namespace cuth {

#ifndef CUTH_CHEB_MINB32
#define CUTH_CHEB_MINB32 8
#endif
#define CUTH_CHEB_NC 1   // columns per thread of the z-marching stencil (2 and 4 measured slower, _work sweep)

// Where the fp32-arithmetic operator takes its off-diagonal entries from: A2 (fp32) or A3 (fp16
// times a power-of-two scale, promoted to fp32 on load: "arithmetic decoupling", Alg. 4).
struct MatF32 {
  // f1..f3 are the aligned per-diagonal copies: an even index is an 8-byte aligned pair, one load
  static __device__ __forceinline__ float2 p1(const DiaDev& A, int64_t i, float) { return *reinterpret_cast<const float2*>(A.f1 + i); }
  static __device__ __forceinline__ float2 p2(const DiaDev& A, int64_t i, float) { return *reinterpret_cast<const float2*>(A.f2 + i); }
  static __device__ __forceinline__ float2 p3(const DiaDev& A, int64_t i, float) { return *reinterpret_cast<const float2*>(A.f3 + i); }
  static __device__ __forceinline__ float inv(const DiaDev&) { return 1.f; }
  static __device__ __forceinline__ float e1(const DiaDev& A, int64_t i, float) { return A.f1[i]; }
  static __device__ __forceinline__ float e2(const DiaDev& A, int64_t i, float) { return A.f2[i]; }
  static __device__ __forceinline__ float e3(const DiaDev& A, int64_t i, float) { return A.f3[i]; }
  // pointer form (kernels that walk a column bump one pointer per diagonal instead of re-deriving indices)
  using elem = float;
  static __device__ __forceinline__ const elem* d1(const DiaDev& A) { return A.f1; }
  static __device__ __forceinline__ const elem* d2(const DiaDev& A) { return A.f2; }
  static __device__ __forceinline__ const elem* d3(const DiaDev& A) { return A.f3; }
  static __device__ __forceinline__ float ld(const elem* p, float) { return *p; }
  static __device__ __forceinline__ float2 ldp(const elem* p, float) { return *reinterpret_cast<const float2*>(p); }   // p at an even element
};
struct MatF16 {
  // the three fp16 arrays are this library's own 256-B aligned copies, so an even index is a 4-byte
  // aligned pair: one half2 load per pair of x-neighbours
  static __device__ __forceinline__ float2 pair(const __half* p, int64_t i, float s) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(p + i));
    return make_float2(f.x * s, f.y * s);
  }
  static __device__ __forceinline__ float2 p1(const DiaDev& A, int64_t i, float s) { return pair(A.h1, i, s); }
  static __device__ __forceinline__ float2 p2(const DiaDev& A, int64_t i, float s) { return pair(A.h2, i, s); }
  static __device__ __forceinline__ float2 p3(const DiaDev& A, int64_t i, float s) { return pair(A.h3, i, s); }
  static __device__ __forceinline__ float inv(const DiaDev& A) { return (float)A.h_scale[2]; }
  static __device__ __forceinline__ float e1(const DiaDev& A, int64_t i, float s) { return __half2float(A.h1[i]) * s; }
  static __device__ __forceinline__ float e2(const DiaDev& A, int64_t i, float s) { return __half2float(A.h2[i]) * s; }
  static __device__ __forceinline__ float e3(const DiaDev& A, int64_t i, float s) { return __half2float(A.h3[i]) * s; }
  using elem = __half;
  static __device__ __forceinline__ const elem* d1(const DiaDev& A) { return A.h1; }
  static __device__ __forceinline__ const elem* d2(const DiaDev& A) { return A.h2; }
  static __device__ __forceinline__ const elem* d3(const DiaDev& A) { return A.h3; }
  static __device__ __forceinline__ float ld(const elem* p, float s) { return __half2float(*p) * s; }
  static __device__ __forceinline__ float2 ldp(const elem* p, float s) {          // p at an even element
    const float2 f = __half22float2(*reinterpret_cast<const __half2*>(p));
    return make_float2(f.x * s, f.y * s);
  }
};

// One row of A v with v stored as VT and arithmetic in T (T = double: A1 standard form; T = float: A2
// difference form, DESIGN.md R-F3), flat traversal.
template <class VT, class T, class M>
__device__ __forceinline__ T row_t(const DiaDev& A, const VT* __restrict__ v, int64_t i, T vi, float ms) {
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = i + np < n, lo3 = i >= np;
  if (sizeof(T) == 8) {
    T acc = (T)A.d0[i] * vi;
    acc += (T)(up1 ? A.d1[i] : 0.0) * (T)(up1 ? v[i + 1] : (VT)0);
    acc += (T)(lo1 ? A.d1[i - 1] : 0.0) * (T)(lo1 ? v[i - 1] : (VT)0);
    acc += (T)(up2 ? A.d2[i] : 0.0) * (T)(up2 ? v[i + nx] : (VT)0);
    acc += (T)(lo2 ? A.d2[i - nx] : 0.0) * (T)(lo2 ? v[i - nx] : (VT)0);
    acc += (T)(up3 ? A.d3[i] : 0.0) * (T)(up3 ? v[i + np] : (VT)0);
    acc += (T)(lo3 ? A.d3[i - np] : 0.0) * (T)(lo3 ? v[i - np] : (VT)0);
    return acc;
  } else {
    const unsigned z = (unsigned)i / (unsigned)np;
    T acc = (T)A.s_layer[z] * vi;
    acc += (T)(up1 ? M::e1(A, i, ms) : 0.f) * ((T)(up1 ? v[i + 1] : (VT)vi) - vi);
    acc += (T)(lo1 ? M::e1(A, i - 1, ms) : 0.f) * ((T)(lo1 ? v[i - 1] : (VT)vi) - vi);
    acc += (T)(up2 ? M::e2(A, i, ms) : 0.f) * ((T)(up2 ? v[i + nx] : (VT)vi) - vi);
    acc += (T)(lo2 ? M::e2(A, i - nx, ms) : 0.f) * ((T)(lo2 ? v[i - nx] : (VT)vi) - vi);
    acc += (T)(up3 ? M::e3(A, i, ms) : 0.f) * ((T)(up3 ? v[i + np] : (VT)vi) - vi);
    acc += (T)(lo3 ? M::e3(A, i - np, ms) : 0.f) * ((T)(lo3 ? v[i - np] : (VT)vi) - vi);
    return acc;
  }
}

// f(i, v_i, (A v)_i) for every row; traversal as in apply_A (flat, or z-marching with the plane
// neighbours in registers).
template <class VT, class T, class M, class F>
__device__ __forceinline__ void apply_A_t(const DiaDev& A, const VT* __restrict__ v, F&& f) {
  const float ms = M::inv(A);
  if (!A.zmarch) {
    CUTH_TILE_LOOP(A.n) {
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * kThreads;
        if (i < A.n) {
          const T vi = (T)v[i];
          f(i, vi, row_t<VT, T, M>(A, v, i, vi, ms));
        }
      }
    }
    return;
  }
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
    T v_lo = (T)0, v_c = (T)v[c], a3l = (T)0;
#pragma unroll 2
    for (int z = 0; z < nz; ++z) {
      const int64_t i = c + (int64_t)z * np;
      const bool up3 = z + 1 < nz;
      const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx;
      T acc, a3u, v_hi;
      if (sizeof(T) == 8) {
        const T a0 = (T)A.d0[i];
        const T a1u = (T)(up1 ? A.d1[i] : 0.0), a1l = (T)(lo1 ? A.d1[i - 1] : 0.0);
        const T a2u = (T)(up2 ? A.d2[i] : 0.0), a2l = (T)(lo2 ? A.d2[i - nx] : 0.0);
        a3u = (T)(up3 ? A.d3[i] : 0.0);
        v_hi = up3 ? (T)v[i + np] : (T)0;
        const T v1u = up1 ? (T)v[i + 1] : (T)0, v1l = lo1 ? (T)v[i - 1] : (T)0;
        const T v2u = up2 ? (T)v[i + nx] : (T)0, v2l = lo2 ? (T)v[i - nx] : (T)0;
        acc = a0 * v_c;
        acc += a1u * v1u; acc += a1l * v1l; acc += a2u * v2u; acc += a2l * v2l;
        acc += a3u * v_hi; acc += a3l * v_lo;
      } else {
        const T a1u = (T)(up1 ? M::e1(A, i, ms) : 0.f), a1l = (T)(lo1 ? M::e1(A, i - 1, ms) : 0.f);
        const T a2u = (T)(up2 ? M::e2(A, i, ms) : 0.f), a2l = (T)(lo2 ? M::e2(A, i - nx, ms) : 0.f);
        a3u = (T)(up3 ? M::e3(A, i, ms) : 0.f);
        v_hi = up3 ? (T)v[i + np] : v_c;
        const T v1u = up1 ? (T)v[i + 1] : v_c, v1l = lo1 ? (T)v[i - 1] : v_c;
        const T v2u = up2 ? (T)v[i + nx] : v_c, v2l = lo2 ? (T)v[i - nx] : v_c;
        acc = (T)A.s_layer[z] * v_c;
        acc += a1u * (v1u - v_c); acc += a1l * (v1l - v_c);
        acc += a2u * (v2u - v_c); acc += a2l * (v2l - v_c);
        acc += a3u * (v_hi - v_c); acc += a3l * ((z > 0 ? v_lo : v_c) - v_c);
      }
      f(i, v_c, acc);
      v_lo = v_c; v_c = v_hi; a3l = a3u;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Alg. 3 with d and r_c eliminated.  With Z_j = d_0 + ... + d_{j-1} (Z_0 = 0, Z_1 = d_0 = r/theta, z = Z_k) the
// algorithm's own identities d_i = Z_{i+1} - Z_i and r_c = r - A Z_{i+1} (lines 6, 8) turn line 10 into
//     Z_{i+2} = Z_{i+1} + c1_i (Z_{i+1} - Z_i) + c2_i (r - A Z_{i+1}),      i = 0 .. k-2,
// the same k-1 stencil passes, but a pass now reads Z_{i+1} (stencil), Z_i and r at its own cell and writes
// Z_{i+2} over Z_i (in place: only the own cell of Z_i is ever read): M + 4s bytes per row instead of M + 6s
// (s = sizeof(T)), and the residual is formed directly instead of by recurrence.  Two buffers Z[0], Z[1]
// (Ctx.cd), named by the `old` / `cur` kernel arguments: the stencil input is Z[cur], the old iterate / output is
// Z[old]; the host schedule (cheb_schedule) swaps them after every pass.  In fp32 mode the first pass also
// leaves an fp32 copy of r (Ctx.crc) for the later passes.
//
// First pass (i = 0): Z_1 = r/theta formed on the fly (A Z_1 = (A r)/theta), Z_2 = Z_1 + c1_0 Z_1 + c2_0 (r - A Z_1).
template <class T, class M>
__global__ void __launch_bounds__(kThreads, sizeof(T) == 4 ? CUTH_CHEB_MINB32 : 4) k_cheb_first(const Ctx* __restrict__ ctxp) {
  const Ctx c = *ctxp;
  const T inv_theta = (T)c.cheb_inv_theta, c1 = (T)ctxp->cheb_c1[0], c2 = (T)ctxp->cheb_c2[0];
  T* __restrict__ z1 = (T*)c.cd[1];
  T* __restrict__ z2 = (T*)c.cd[0];
  T* __restrict__ r32 = (T*)c.crc;
  apply_A_t<double, T, M>(c.A, c.r, [&](int64_t i, T ri, T Ar) {
    const T Z1 = ri * inv_theta;                 // lines 4, 6
    const T res = ri - Ar * inv_theta;           // r - A Z_1 (lines 7-8)
    z1[i] = Z1;
    z2[i] = Z1 + c1 * Z1 + c2 * res;             // line 10, then line 6 of the next pass
    if (sizeof(T) == 4) r32[i] = ri;
  });
}

// Passes 0 < i < k-2.
template <class T, class M>
__global__ void __launch_bounds__(kThreads, sizeof(T) == 4 ? CUTH_CHEB_MINB32 : 4) k_cheb_mid(const Ctx* __restrict__ ctxp, int step,
                                                                                              int old, int cur) {
  const Ctx c = *ctxp;
  const T c1 = (T)ctxp->cheb_c1[step], c2 = (T)ctxp->cheb_c2[step];
  const T* __restrict__ zcur = (const T*)ctxp->cd[cur];
  T* __restrict__ zold = (T*)ctxp->cd[old];
  const T* __restrict__ r32 = (const T*)c.crc;
  apply_A_t<T, T, M>(c.A, zcur, [&](int64_t i, T zi, T Az) {
    const T ri = sizeof(T) == 4 ? r32[i] : (T)c.r[i];
    zold[i] = zi + c1 * (zi - zold[i]) + c2 * (ri - Az);
  });
}

// The same middle step for T = float on large planes with even nx: each thread owns TWO x-adjacent columns,
// so the vectors Z_{i+1}, Z_i, r move as 8-byte float2 (every row start is even => 8-byte aligned), the +-1
// neighbours of the pair are each other (registers), and a thread keeps twice the bytes in flight -- the
// 4-byte version is latency-bound (profiles/r1c_cfg3_cheb_mixed.md).  Matrix entries stay scalar loads: the
// packed diagonals D2, D3 start at odd elements (R-G5b).  Tile = (2 ZTX) x ZTY columns per CTA.
template <class M>
__global__ void __launch_bounds__(kThreads, 6) k_cheb_mid_f32x2(const Ctx* __restrict__ ctxp, int step, int old, int cur) {
  const Ctx c = *ctxp;
  const DiaDev& A = c.A;
  const float c1 = (float)ctxp->cheb_c1[step], c2 = (float)ctxp->cheb_c2[step];
  const float* __restrict__ din = (const float*)ctxp->cd[cur];                // Z_{i+1}: stencil input
  float* __restrict__ zold = (float*)ctxp->cd[old];                           // Z_i in, Z_{i+2} out (in place)
  const float* __restrict__ r32 = (const float*)c.crc;
  const int tx = threadIdx.x % ZTX, ty = threadIdx.x / ZTX;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + 2 * ZTX - 1) / (2 * ZTX), tiles_y = (nyi + ZTY - 1) / ZTY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  auto ld2 = [](const float* p) { return *reinterpret_cast<const float2*>(p); };
  const float ms = M::inv(A);
  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x = bx * 2 * ZTX + 2 * tx, y = by * ZTY + ty;
    if (x >= nxi || y >= nyi) continue;                 // nx even: x + 1 < nx as well
    const int64_t c0 = x + nx * (int64_t)y;
    float2 v_lo = make_float2(0.f, 0.f), v_c = ld2(din + c0), a3l = make_float2(0.f, 0.f);
#pragma unroll 2
    for (int z = 0; z < nz; ++z) {
      const int64_t i = c0 + (int64_t)z * np;
      const bool up3 = z + 1 < nz, up2 = i + nx < n, lo2 = i >= nx, lo1 = i >= 1, up1 = i + 2 < n;
      // entries of the pair (i, i+1); the element i+1 of D1 couples to i+2, which may not exist
      const float f1l = lo1 ? M::e1(A, i - 1, ms) : 0.f;
      float2 f1p = up1 ? M::p1(A, i, ms) : make_float2(M::e1(A, i, ms), 0.f);
      const float f1a = f1p.x, f1b = f1p.y;
      const float2 z2 = make_float2(0.f, 0.f);
      const float2 f2u = up2 ? M::p2(A, i, ms) : z2, f2l = lo2 ? M::p2(A, i - nx, ms) : z2;
      const float f2u0 = f2u.x, f2u1 = f2u.y, f2l0 = f2l.x, f2l1 = f2l.y;
      const float2 a3u = up3 ? M::p3(A, i, ms) : z2;
      const float2 v_hi = up3 ? ld2(din + i + np) : v_c;
      const float2 v2u = up2 ? ld2(din + i + nx) : v_c, v2l = lo2 ? ld2(din + i - nx) : v_c;
      const float vl = lo1 ? din[i - 1] : v_c.x, vr = up1 ? din[i + 2] : v_c.y;
      const float2 rv = ld2(r32 + i), zo = ld2(zold + i);
      const float s = (float)A.s_layer[z];
      float a0 = s * v_c.x, a1 = s * v_c.y;
      a0 += f1a * (v_c.y - v_c.x);   a1 += f1a * (v_c.x - v_c.y);
      a0 += f1l * (vl - v_c.x);      a1 += f1b * (vr - v_c.y);
      a0 += f2u0 * (v2u.x - v_c.x);  a1 += f2u1 * (v2u.y - v_c.y);
      a0 += f2l0 * (v2l.x - v_c.x);  a1 += f2l1 * (v2l.y - v_c.y);
      a0 += a3u.x * (v_hi.x - v_c.x); a1 += a3u.y * (v_hi.y - v_c.y);
      a0 += a3l.x * (v_lo.x - v_c.x); a1 += a3l.y * (v_lo.y - v_c.y);    // a3l = 0 at z = 0
      *reinterpret_cast<float2*>(zold + i) = make_float2(v_c.x + c1 * (v_c.x - zo.x) + c2 * (rv.x - a0),
                                                         v_c.y + c1 * (v_c.y - zo.y) + c2 * (rv.y - a1));
      v_lo = v_c; v_c = v_hi; a3l = a3u;
    }
  }
}

// Last pass (i = k-2): z = Z_k in fp64 for the outer loop, and rho = r.z (Alg. 1 lines 10-11).
template <class T, class M>
__global__ void __launch_bounds__(kThreads, sizeof(T) == 4 ? 6 : 4) k_cheb_last(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials,
                                                        int step, int old, int cur) {
  __shared__ double smem[32];
  __shared__ int s_flag;
  const Ctx c = *ctxp;
  const T c1 = (T)ctxp->cheb_c1[step], c2 = (T)ctxp->cheb_c2[step];
  const T* __restrict__ zcur = (const T*)ctxp->cd[cur];
  const T* __restrict__ zold = (const T*)ctxp->cd[old];
  double acc[1] = {0.0};
  apply_A_t<T, T, M>(c.A, zcur, [&](int64_t i, T zi, T Az) {
    const double rd = c.r[i];
    const double zk = (double)(zi + c1 * (zi - zold[i]) + c2 * ((T)rd - Az));
    c.cz[i] = zk;
    acc[0] = fma(rd, zk, acc[0]);
  });
  if (grid_sum_last_block<1>(acc, partials + 3 * kMaxBlocks, &ctl->ticket[5], smem, &s_flag) && threadIdx.x == 0) {
    const double rho_new = acc[0];
    ctl->beta = ctl->beta_zero ? 0.0 : rho_new / ctl->rho;     // Alg. 1 line 11 (line 3 when restarting)
    ctl->rho = rho_new;
    ctl->beta_zero = 0;
    if (!(rho_new == rho_new) || rho_new <= 0.0) ctl->status = CUTH_SOLVE_BREAKDOWN;   // q(A) not SPD: bad interval
  }
}

// ---------------------------------------------------------------------------------------------
// Lanczos on unnormalised vectors u_j (v_j = s_j u_j, s_j = 1/||u_j||):
//   L1: t = s_j A u_j - beta_{j-1} s_{j-1} u_{j-1},  alpha_j = s_j (t . u_j)
//   L2: u_{j+1} = t - alpha_j s_j u_j (overwrites u_{j-1}),  beta_j = ||u_{j+1}||
struct LanczosScal { double s_cur, s_prev, beta_prev, alpha; double out_alpha[128], out_beta[128]; int j, pad; unsigned ticket[2]; };

__global__ void __launch_bounds__(kThreads, 4) k_lanczos_1(DiaDev A, const double* __restrict__ u_cur,
                                                         const double* __restrict__ u_prev, double* __restrict__ t,
                                                         LanczosScal* sc, double* partials) {
  __shared__ double smem[32];
  __shared__ int s_flag;
  const double s_cur = sc->s_cur, cprev = sc->beta_prev * sc->s_prev;
  double acc[1] = {0.0};
  apply_A<OP_FP64>(A, u_cur, [&](int64_t i, double ui, double Au) {
    const double ti = s_cur * Au - cprev * u_prev[i];
    t[i] = ti;
    acc[0] = fma(ti, ui, acc[0]);
  });
  if (grid_sum_last_block<1>(acc, partials, &sc->ticket[0], smem, &s_flag) && threadIdx.x == 0)
    sc->alpha = s_cur * acc[0];
}

// The paper's variant of L1: fp32 vectors, the fixed-FP32 SpMV of Alg. 2 on the fp32 copy A2 (all four
// diagonals, standard form), fp32 arithmetic; per-thread sums in fp32, widened only for the fixed-order grid reduction.
__global__ void __launch_bounds__(kThreads, 4) k_lanczos_1_f32(DiaDev A, const float* __restrict__ u_cur,
                                                             const float* __restrict__ u_prev, float* __restrict__ t,
                                                             LanczosScal* sc, double* partials) {
  __shared__ double smem[32];
  __shared__ int s_flag;
  const float s_cur = (float)sc->s_cur, cprev = (float)(sc->beta_prev * sc->s_prev);
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  float facc = 0.f;
  CUTH_TILE_LOOP(n) {
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      const int64_t i = base + threadIdx.x + k * kThreads;
      if (i < n) {
        const float ui = u_cur[i];
        float au = A.f0[i] * ui;
        if (i + 1 < n) au = fmaf(A.f1[i], u_cur[i + 1], au);
        if (i >= 1) au = fmaf(A.f1[i - 1], u_cur[i - 1], au);
        if (i + nx < n) au = fmaf(A.f2[i], u_cur[i + nx], au);
        if (i >= nx) au = fmaf(A.f2[i - nx], u_cur[i - nx], au);
        if (i + np < n) au = fmaf(A.f3[i], u_cur[i + np], au);
        if (i >= np) au = fmaf(A.f3[i - np], u_cur[i - np], au);
        const float ti = s_cur * au - cprev * u_prev[i];
        t[i] = ti;
        facc = fmaf(ti, ui, facc);
      }
    }
  }
  double acc[1] = {(double)facc};
  if (grid_sum_last_block<1>(acc, partials, &sc->ticket[0], smem, &s_flag) && threadIdx.x == 0)
    sc->alpha = (double)(s_cur * (float)acc[0]);
}

template <class V>
__global__ void __launch_bounds__(kThreads) k_lanczos_2(int64_t n, const V* __restrict__ u_cur,
                                                       const V* __restrict__ t, V* __restrict__ u_next,
                                                       LanczosScal* sc, double* partials) {
  __shared__ double smem[32];
  __shared__ int s_flag;
  const V a = (V)(sc->alpha * sc->s_cur);
  V vacc = (V)0;
  CUTH_TILE_LOOP(n) {
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      const int64_t i = base + threadIdx.x + k * kThreads;
      if (i < n) {
        const V v = t[i] - a * u_cur[i];
        u_next[i] = v;
        vacc = v * v + vacc;
      }
    }
  }
  double acc[1] = {(double)vacc};
  if (grid_sum_last_block<1>(acc, partials + kMaxBlocks, &sc->ticket[1], smem, &s_flag) && threadIdx.x == 0) {
    const double beta = sqrt(acc[0]);
    const int j = sc->j;
    sc->out_alpha[j] = sc->alpha;
    sc->out_beta[j] = beta;
    sc->beta_prev = beta;
    sc->s_prev = sc->s_cur;
    sc->s_cur = beta > 0.0 ? 1.0 / beta : 0.0;
    sc->j = j + 1;
  }
}

// u_0 = v0, u_{-1} = 0, s_0 = 1/||v0||; also the Gershgorin bound max_i sum_j |a_ij| (into out_beta[127]).
template <class V>
__global__ void __launch_bounds__(kThreads) k_lanczos_init(DiaDev A, const double* __restrict__ v0,
                                                          V* __restrict__ u_cur, V* __restrict__ u_prev,
                                                          LanczosScal* sc, double* partials) {
  __shared__ double smem[2 * 32];
  __shared__ int s_flag;
  double acc[1] = {0.0};
  double gmax = 0.0;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  CUTH_TILE_LOOP(n) {
#pragma unroll
    for (int k = 0; k < kRows; ++k) {
      const int64_t i = base + threadIdx.x + k * kThreads;
      if (i < n) {
        const V vv = (V)v0[i];
        const double v = (double)vv;
        u_cur[i] = vv;
        u_prev[i] = (V)0;
        acc[0] = fma(v, v, acc[0]);
        double g = fabs(A.d0[i]);
        if (i + 1 < n) g += fabs(A.d1[i]);
        if (i >= 1) g += fabs(A.d1[i - 1]);
        if (i + nx < n) g += fabs(A.d2[i]);
        if (i >= nx) g += fabs(A.d2[i - nx]);
        if (i + np < n) g += fabs(A.d3[i]);
        if (i >= np) g += fabs(A.d3[i - np]);
        gmax = fmax(gmax, g);
      }
    }
  }
  // max over the grid: positive doubles order like their bit patterns
  for (int o = 16; o > 0; o >>= 1) gmax = fmax(gmax, __shfl_xor_sync(0xffffffffu, gmax, o));
  if ((threadIdx.x & 31) == 0) atomicMax((unsigned long long*)&sc->out_beta[127], (unsigned long long)__double_as_longlong(gmax));
  if (grid_sum_last_block<1>(acc, partials, &sc->ticket[0], smem, &s_flag) && threadIdx.x == 0) {
    sc->s_cur = acc[0] > 0.0 ? 1.0 / sqrt(acc[0]) : 0.0;
    sc->s_prev = 0.0; sc->beta_prev = 0.0; sc->j = 0;
  }
}

}  // namespace cuth
