// cuth_fused.cuh -- the two-kernel PCG iteration for large planes ("fused path").
//
//   K1 = k_fused_pspmv : p' = M^-1 r + beta p   (Alg. 1 line 12, with line 10 recomputed)
//                        x += alpha_prev p      (Alg. 1 line 8, deferred by one kernel)
//                        mu = A p', p'.mu       (Alg. 1 line 6 and the denominator of line 7)
//   K2 = k_fused_update: r -= alpha mu, z = M^-1 r, r.z, ||r||^2   (lines 9-11)
//
// Algorithmic traffic per row and iteration, fp64 operator: K1 = E/N matrix elements + r, p, x read +
// p', mu, x written (8m + 48 B; M^-1 comes from the D0 the SpMV reads anyway, one plane early), K2 = r, mu,
// 1/D0 read + r written (32 B): 8m + 80 B, 8 B below the 8m + 88 floor SURVEY.md §8(d) counts.  fp32-stored
// operator (early stage): D0 is not part of it, K1 reads 1/D0: 4(m-1) + 56 + 32 B.
//
// K1 walks the grid like zmarch_apply (a CTA owns a TX x TY tile of the x-y plane, a thread owns one
// column and marches in z), but the vector it multiplies is produced on the fly: each thread forms
// p' for its own cell one plane ahead, the tile perimeter (halo) is recomputed by the first
// 2(TX+TY) threads from r, 1/D0, p (L2 hits: the neighbouring CTA streams the same lines), and one
// plane of p' (tile + halo) is exchanged through double-buffered shared memory, one barrier per
// plane.  p is ping-ponged between two buffers because neighbouring CTAs read the old p of cells
// this CTA overwrites.
#pragma once
#include "cuth_kernels.cuh"

namespace cuth {

constexpr int FTX = 32, FTY = 8;     // FTX * FTY == kThreads
static_assert(FTX * FTY == kThreads, "tile must match the block size");
constexpr int kHalo = 2 * FTX + 2 * FTY;
constexpr int kHaloPerWarp = (kHalo + kThreads / 32 - 1) / (kThreads / 32);

// 1 / d for a positive normal d (a main-diagonal entry, R-G2), to within an ulp: hardware seed (>= 20 bits)
// and two Newton steps; no special cases, hence no slow-path call and no extra registers.
__device__ __forceinline__ double rcp_diag(double d) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
  double e = fma(-d, y, 1.0);
  y = fma(y, e, y);
  e = fma(-d, y, 1.0);
  return fma(y, e, y);
}

template <bool MIXED>
__device__ __forceinline__ void fused_pspmv_body(const Ctx& c, const double* __restrict__ p_in,
                                                 double* __restrict__ p_out, const double beta,
                                                 const double xalpha, double (*sp)[FTY + 2][FTX + 2],
                                                 double& dot) {
  const DiaDev& A = c.A;
  const int tx = threadIdx.x % FTX, ty = threadIdx.x / FTX;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + FTX - 1) / FTX, tiles_y = (nyi + FTY - 1) / FTY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const bool jac = c.jacobi != 0;
  const double* __restrict__ zs = c.cheb ? c.cz : c.r;     // Chebyshev: z = q(A) r is a stored vector
  const bool do_x = xalpha != 0.0;

  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x = bx * FTX + tx, y = by * FTY + ty;
    const bool own = x < nxi && y < nyi;
    const int64_t col = own ? x + nx * (int64_t)y : 0;
    // halo role of this thread: the 2(TX+TY) perimeter cells of a plane are dealt evenly to the warps
    // (kHaloPerWarp lanes of each warp take one cell), so that no warp reaches the barrier late.
    int hx = -1, hy = -1, hr = 0, hc = 0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int h = lane < kHaloPerWarp ? wid * kHaloPerWarp + lane : kHalo;
    if (h < FTX)                { hx = bx * FTX + h;            hy = by * FTY - 1;   hr = 0;        hc = h + 1; }
    else if (h < 2 * FTX)       { hx = bx * FTX + (h - FTX);    hy = by * FTY + FTY; hr = FTY + 1;  hc = h - FTX + 1; }
    else if (h < 2 * FTX + FTY) { hx = bx * FTX - 1;            hy = by * FTY + (h - 2 * FTX);       hr = h - 2 * FTX + 1;       hc = 0; }
    else if (h < kHalo)         { hx = bx * FTX + FTX;          hy = by * FTY + (h - 2 * FTX - FTY); hr = h - 2 * FTX - FTY + 1; hc = FTX + 1; }
    const bool halo_role = h < kHalo;
    const bool halo_in = halo_role && hx >= 0 && hx < nxi && hy >= 0 && hy < nyi;
    const int64_t hcol = halo_in ? hx + nx * (int64_t)hy : 0;

    __syncthreads();                       // previous tile's planes are dead
    double pn_lo = 0.0, pn_c = 0.0, a3l = 0.0;
    double dnx = 1.0;                      // fp64 operator: D0 of the plane p' is being formed for (M, then SpMV)
    {   // plane 0 of p'
      double ro = 0.0, dio = 1.0, po = 0.0, xo = 0.0, rh = 0.0, dih = 1.0, ph = 0.0;
      if (own) {
        ro = zs[col]; po = p_in[col];
        if (MIXED) { if (jac) dio = (double)A.dinv32[col]; } else { dnx = A.d0[col]; }
        if (do_x) xo = c.x[col];
      }
      if (halo_in) { rh = zs[hcol]; ph = p_in[hcol]; if (jac) dih = MIXED ? (double)A.dinv32[hcol] : A.d0[hcol]; }
      if (own) {
        pn_c = fma(beta, po, MIXED ? ro * dio : (jac ? ro * rcp_diag(dnx) : ro));
        p_out[col] = pn_c;
        if (do_x) c.x[col] = fma(xalpha, po, xo);
      }
      sp[0][ty + 1][tx + 1] = pn_c;
      if (halo_role) sp[0][hr][hc] = halo_in ? fma(beta, ph, MIXED ? rh * dih : rh * rcp_diag(dih)) : 0.0;
    }

    for (int z = 0; z < nz; ++z) {
      const int cur = z & 1, nxt = cur ^ 1;
      const int64_t i = col + (int64_t)z * np;
      const bool up3 = z + 1 < nz;
      // ---- 1. every global load of this step, issued back to back: matrix operands of row i,
      //         vector operands of plane z+1 (own cell and halo cell)
      double a0 = 0.0, a1u = 0.0, a1l = 0.0, a2u = 0.0, a2l = 0.0, a3u = 0.0;
      double ro = 0.0, dio = 1.0, po = 0.0, xo = 0.0, rh = 0.0, dih = 1.0, ph = 0.0;
      if (own) {
        const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx;
        if (!MIXED) {
          a0 = dnx;                                // loaded during the previous step
          a1u = up1 ? A.d1[i] : 0.0;  a1l = lo1 ? A.d1[i - 1] : 0.0;
          a2u = up2 ? A.d2[i] : 0.0;  a2l = lo2 ? A.d2[i - nx] : 0.0;
          a3u = up3 ? A.d3[i] : 0.0;
        } else {
          a1u = up1 ? (double)A.f1[i] : 0.0;  a1l = lo1 ? (double)A.f1[i - 1] : 0.0;
          a2u = up2 ? (double)A.f2[i] : 0.0;  a2l = lo2 ? (double)A.f2[i - nx] : 0.0;
          a3u = up3 ? (double)A.f3[i] : 0.0;
        }
        if (up3) {
          const int64_t j = i + np;
          ro = zs[j]; po = p_in[j];
          if (MIXED) { if (jac) dio = (double)A.dinv32[j]; } else { dnx = A.d0[j]; }
          if (do_x) xo = c.x[j];
        }
      }
      if (up3 && halo_in) {
        const int64_t j = hcol + (int64_t)(z + 1) * np;
        rh = zs[j]; ph = p_in[j];
        if (jac) dih = MIXED ? (double)A.dinv32[j] : A.d0[j];
      }
      // ---- 2. plane z of p' (written during the previous step) is complete; the loads above fly
      //         while the CTA waits here
      __syncthreads();
      // ---- 3. plane z+1 of p': own cell (kept in a register) and halo cell, into the other buffer
      double pn_hi = 0.0;
      if (up3) {
        if (own) {
          pn_hi = fma(beta, po, MIXED ? ro * dio : (jac ? ro * rcp_diag(dnx) : ro));
          p_out[i + np] = pn_hi;
          if (do_x) c.x[i + np] = fma(xalpha, po, xo);
        }
        sp[nxt][ty + 1][tx + 1] = pn_hi;
        if (halo_role) sp[nxt][hr][hc] = halo_in ? fma(beta, ph, MIXED ? rh * dih : rh * rcp_diag(dih)) : 0.0;
      }
      // ---- 4. row i of mu = A p'
      if (own) {
        const double v1l = sp[cur][ty + 1][tx], v1u = sp[cur][ty + 1][tx + 2];
        const double v2l = sp[cur][ty][tx + 1], v2u = sp[cur][ty + 2][tx + 1];
        double acc;
        if (!MIXED) {
          acc = a0 * pn_c;
          acc = fma(a1u, v1u, acc); acc = fma(a1l, v1l, acc);
          acc = fma(a2u, v2u, acc); acc = fma(a2l, v2l, acc);
          acc = fma(a3u, pn_hi, acc); acc = fma(a3l, pn_lo, acc);
        } else {
          acc = A.s_layer[z] * pn_c;
          acc = fma(a1u, v1u - pn_c, acc); acc = fma(a1l, v1l - pn_c, acc);
          acc = fma(a2u, v2u - pn_c, acc); acc = fma(a2l, v2l - pn_c, acc);
          acc = fma(a3u, pn_hi - pn_c, acc); acc = fma(a3l, pn_lo - pn_c, acc);
        }
        c.mu[i] = acc;
        dot = fma(pn_c, acc, dot);
      }
      pn_lo = pn_c; pn_c = pn_hi; a3l = a3u;
    }
  }
}

// K1.  ctl->pcur selects which of the two p buffers holds the current direction.
__global__ void __launch_bounds__(kThreads, 4) k_fused_pspmv(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials) {
  __shared__ double sp[2][FTY + 2][FTX + 2];
  __shared__ double smem[32];
  __shared__ int s_flag;
  if (ctl->halt) return;                     // unrolled graph body: this pass is over
  const Ctx c = *ctxp;
  const int pcur = ctl->pcur;
  const double* p_in = pcur ? c.p2 : c.p;
  double* p_out = pcur ? c.p : c.p2;
  const double beta = ctl->beta, xalpha = ctl->xalpha;
  double acc[1] = {0.0};
  if (ctl->stage == 0) fused_pspmv_body<true>(c, p_in, p_out, beta, xalpha, sp, acc[0]);
  else fused_pspmv_body<false>(c, p_in, p_out, beta, xalpha, sp, acc[0]);
  if (grid_sum_last_block<1>(acc, partials, &ctl->ticket[1], smem, &s_flag) && threadIdx.x == 0) {
    ctl->pcur = pcur ^ 1;
    policy_after_spmv(ctl, acc[0], true, &c);   // Alg. 1 line 7; x += alpha p deferred to the next K1 (or to K2: xnow)
  }
}

// Applies the deferred x += alpha p before a true-residual evaluation (k_true_resid's epilogue then
// clears ctl->xalpha; k_finalize applies whatever is still pending at the end of the solve).
__global__ void __launch_bounds__(kThreads) k_flush_x(const Ctx* __restrict__ ctxp, Ctl* ctl) {
  const Ctx c = *ctxp;
  const double xalpha = ctl->xalpha;
  if (xalpha != 0.0) {
    const double* p = ctl->pcur ? c.p2 : c.p;
    CUTH_TILE_LOOP(c.A.n) {
#pragma unroll
      for (int k = 0; k < kRows; ++k) {
        const int64_t i = base + threadIdx.x + k * kThreads;
        if (i < c.A.n) c.x[i] = fma(xalpha, p[i], c.x[i]);
      }
    }
  }
}

}  // namespace cuth
