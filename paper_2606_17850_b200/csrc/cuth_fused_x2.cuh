// cuth_fused_x2.cuh -- K1 (k_fused_pspmv, see cuth_fused.cuh) with TWO x-adjacent columns per thread, used
// when nx is even.  Same algorithm, same buffers, same reduction and epilogue; what changes is the
// instruction stream: the per-row index / predicate / halo bookkeeping is shared by two rows, the vectors
// r, 1/D0, p, x, p', mu move as 16-byte double2 (every row starts at an even index, so they are aligned),
// the +-1 neighbours of the pair are each other (registers), and D0 / D1 pairs are double2 too (their packed
// starts 0 and N are even; D2 and D3 start at odd elements, R-G5b, and stay scalar).  ncu on the one-column
// K1: 230 instructions per row, ALU pipe 38 %, issue slots 48 % busy -- it is instruction-, not byte-bound.
// Tile = 64 x 8 columns per CTA; shared plane 10 x 68 doubles, interior starting at an even column.
#pragma once
#include "cuth_fused.cuh"

namespace cuth {

constexpr int XTX = 64, XTY = 8;                 // columns per CTA tile; 32 x 8 threads
constexpr int XS = XTX + 4;                       // smem row: [pad][left halo][64 interior][right halo][pad]
constexpr int kHaloX2 = 2 * XTX + 2 * XTY;        // 144 perimeter cells per plane
constexpr int kHaloX2PerWarp = kHaloX2 / (kThreads / 32);   // 18 lanes of each warp
static_assert(kHaloX2 % (kThreads / 32) == 0, "halo must divide evenly among the warps");

__device__ __forceinline__ double2 ldd2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ double2 ldf2(const float* p) {       // an aligned pair of floats, promoted
  const float2 f = *reinterpret_cast<const float2*>(p);
  return make_double2((double)f.x, (double)f.y);
}
__device__ __forceinline__ void std2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }

template <bool MIXED>
__device__ __forceinline__ void fused_pspmv_x2_body(const Ctx& c, const double* __restrict__ p_in,
                                                    double* __restrict__ p_out, const double beta,
                                                    const double xalpha, double (*sp)[XTY + 2][XS], double& dot) {
  const DiaDev& A = c.A;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + XTX - 1) / XTX, tiles_y = (nyi + XTY - 1) / XTY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const bool jac = c.jacobi != 0;
  const double* __restrict__ zs = c.cheb ? c.cz : c.r;
  const bool do_x = xalpha != 0.0;
  const int sc0 = 2 + 2 * tx;                     // smem column of the pair's first element (even)

  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x = bx * XTX + 2 * tx, y = by * XTY + ty;
    const bool own = x < nxi && y < nyi;          // nx even: x + 1 < nx too
    const int64_t col = own ? x + nx * (int64_t)y : 0;
    // halo role: 18 lanes of each warp take one perimeter cell of the plane
    int hx = -1, hy = -1, hr = 0, hc = 0;
    const int h = tx < kHaloX2PerWarp ? ty * kHaloX2PerWarp + tx : kHaloX2;
    if (h < XTX)                { hx = bx * XTX + h;           hy = by * XTY - 1;   hr = 0;        hc = 2 + h; }
    else if (h < 2 * XTX)       { hx = bx * XTX + (h - XTX);   hy = by * XTY + XTY; hr = XTY + 1;  hc = 2 + h - XTX; }
    else if (h < 2 * XTX + XTY) { hx = bx * XTX - 1;           hy = by * XTY + (h - 2 * XTX);       hr = h - 2 * XTX + 1;       hc = 1; }
    else if (h < kHaloX2)       { hx = bx * XTX + XTX;         hy = by * XTY + (h - 2 * XTX - XTY); hr = h - 2 * XTX - XTY + 1; hc = 2 + XTX; }
    const bool halo_role = h < kHaloX2;
    const bool halo_in = halo_role && hx >= 0 && hx < nxi && hy >= 0 && hy < nyi;
    const int64_t hcol = halo_in ? hx + nx * (int64_t)hy : 0;

    __syncthreads();                              // previous tile's planes are dead
    double pc0 = 0.0, pc1 = 0.0, pl0 = 0.0, pl1 = 0.0, a3l0 = 0.0, a3l1 = 0.0;
    // fp64 operator: the main diagonal of plane z+1 is loaded one step early and serves twice, as M = diag A
    // of Alg. 1 line 10 (z = r / D0 as r * rcp(D0), rcp to within an ulp like the stored 1/D0) and then as the D0 term of the SpMV;
    // 1/D0 is not read at all (8 B/row less).  fp32-stored operator: D0 is not part of it, 1/D0 is read.
    double2 dnx = make_double2(1.0, 1.0);           // D0 of the plane p' is being formed for
    {   // plane 0 of p'
      double2 ro = make_double2(0.0, 0.0), po = ro, xo = ro, dio = make_double2(1.0, 1.0);
      double rh = 0.0, dih = 1.0, ph = 0.0;
      if (own) {
        ro = ldd2(zs + col); po = ldd2(p_in + col);
        if (MIXED) { if (jac) dio = ldf2(A.dinv32 + col); } else { dnx = ldd2(A.d0 + col); }
        if (do_x) xo = ldd2(c.x + col);
      }
      if (halo_in) { rh = zs[hcol]; ph = p_in[hcol]; if (jac) dih = MIXED ? (double)A.dinv32[hcol] : A.d0[hcol]; }
      if (own) {
        const double z0 = MIXED ? ro.x * dio.x : (jac ? ro.x * rcp_diag(dnx.x) : ro.x);
        const double z1 = MIXED ? ro.y * dio.y : (jac ? ro.y * rcp_diag(dnx.y) : ro.y);
        pc0 = fma(beta, po.x, z0); pc1 = fma(beta, po.y, z1);
        std2(p_out + col, pc0, pc1);
        if (do_x) std2(c.x + col, fma(xalpha, po.x, xo.x), fma(xalpha, po.y, xo.y));
      }
      std2(&sp[0][ty + 1][sc0], pc0, pc1);
      if (halo_role) sp[0][hr][hc] = halo_in ? fma(beta, ph, MIXED ? rh * dih : rh * rcp_diag(dih)) : 0.0;
    }

    for (int z = 0; z < nz; ++z) {
      const int cur = z & 1, nxt = cur ^ 1;
      const int64_t i = col + (int64_t)z * np;
      const bool up3 = z + 1 < nz;
      // ---- 1. all global loads of the step
      double a00 = 0.0, a01 = 0.0, a1a = 0.0, a1b = 0.0, a1l = 0.0;
      double a2u0 = 0.0, a2u1 = 0.0, a2l0 = 0.0, a2l1 = 0.0, a3u0 = 0.0, a3u1 = 0.0;
      double2 ro = make_double2(0.0, 0.0), po = ro, xo = ro, dio = make_double2(1.0, 1.0);
      double rh = 0.0, dih = 1.0, ph = 0.0;
      if (own) {
        const bool up1 = i + 2 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx;   // the pair shares up2 / lo2
        if (!MIXED) {
          a00 = dnx.x; a01 = dnx.y;               // loaded during the previous step
          if (up1) { const double2 d1 = ldd2(A.d1 + i); a1a = d1.x; a1b = d1.y; } else { a1a = A.d1[i]; }
          a1l = lo1 ? A.d1[i - 1] : 0.0;
          if (up2) { a2u0 = A.d2[i]; a2u1 = A.d2[i + 1]; }
          if (lo2) { a2l0 = A.d2[i - nx]; a2l1 = A.d2[i + 1 - nx]; }
          if (up3) { a3u0 = A.d3[i]; a3u1 = A.d3[i + 1]; }
        } else {
          if (up1) { const float2 f = *reinterpret_cast<const float2*>(A.f1 + i); a1a = (double)f.x; a1b = (double)f.y; }
          else { a1a = (double)A.f1[i]; }
          a1l = lo1 ? (double)A.f1[i - 1] : 0.0;
          // aligned per-diagonal fp32 copies: every pair is one 8-byte load
          if (up2) { const float2 f = *reinterpret_cast<const float2*>(A.f2 + i); a2u0 = (double)f.x; a2u1 = (double)f.y; }
          if (lo2) { const float2 f = *reinterpret_cast<const float2*>(A.f2 + i - nx); a2l0 = (double)f.x; a2l1 = (double)f.y; }
          if (up3) { const float2 f = *reinterpret_cast<const float2*>(A.f3 + i); a3u0 = (double)f.x; a3u1 = (double)f.y; }
        }
        if (up3) {
          const int64_t j = i + np;
          ro = ldd2(zs + j); po = ldd2(p_in + j);
          if (MIXED) { if (jac) dio = ldf2(A.dinv32 + j); } else { dnx = ldd2(A.d0 + j); }
          if (do_x) xo = ldd2(c.x + j);
        }
      }
      if (up3 && halo_in) {
        const int64_t j = hcol + (int64_t)(z + 1) * np;
        rh = zs[j]; ph = p_in[j];
        if (jac) dih = MIXED ? (double)A.dinv32[j] : A.d0[j];
      }
      // ---- 2. plane z of p' is complete (written during the previous step); the loads fly meanwhile
      __syncthreads();
      // ---- 3. plane z+1 of p'
      double ph0 = 0.0, ph1 = 0.0;
      if (up3) {
        if (own) {
          const double z0 = MIXED ? ro.x * dio.x : (jac ? ro.x * rcp_diag(dnx.x) : ro.x);
          const double z1 = MIXED ? ro.y * dio.y : (jac ? ro.y * rcp_diag(dnx.y) : ro.y);
          ph0 = fma(beta, po.x, z0); ph1 = fma(beta, po.y, z1);
          std2(p_out + i + np, ph0, ph1);
          if (do_x) std2(c.x + i + np, fma(xalpha, po.x, xo.x), fma(xalpha, po.y, xo.y));
        }
        std2(&sp[nxt][ty + 1][sc0], ph0, ph1);
        if (halo_role) sp[nxt][hr][hc] = halo_in ? fma(beta, ph, MIXED ? rh * dih : rh * rcp_diag(dih)) : 0.0;
      }
      // ---- 4. rows i, i+1 of mu = A p'
      if (own) {
        const double vl = sp[cur][ty + 1][sc0 - 1], vr = sp[cur][ty + 1][sc0 + 2];
        const double2 dn = *reinterpret_cast<const double2*>(&sp[cur][ty][sc0]);
        const double2 up = *reinterpret_cast<const double2*>(&sp[cur][ty + 2][sc0]);
        double m0, m1;
        if (!MIXED) {
          m0 = a00 * pc0;                 m1 = a01 * pc1;
          m0 = fma(a1a, pc1, m0);         m1 = fma(a1a, pc0, m1);
          m0 = fma(a1l, vl, m0);          m1 = fma(a1b, vr, m1);
          m0 = fma(a2u0, up.x, m0);       m1 = fma(a2u1, up.y, m1);
          m0 = fma(a2l0, dn.x, m0);       m1 = fma(a2l1, dn.y, m1);
          m0 = fma(a3u0, ph0, m0);        m1 = fma(a3u1, ph1, m1);
          m0 = fma(a3l0, pl0, m0);        m1 = fma(a3l1, pl1, m1);
        } else {
          const double s = A.s_layer[z];
          m0 = s * pc0;                           m1 = s * pc1;
          m0 = fma(a1a, pc1 - pc0, m0);           m1 = fma(a1a, pc0 - pc1, m1);
          m0 = fma(a1l, vl - pc0, m0);            m1 = fma(a1b, vr - pc1, m1);
          m0 = fma(a2u0, up.x - pc0, m0);         m1 = fma(a2u1, up.y - pc1, m1);
          m0 = fma(a2l0, dn.x - pc0, m0);         m1 = fma(a2l1, dn.y - pc1, m1);
          m0 = fma(a3u0, ph0 - pc0, m0);          m1 = fma(a3u1, ph1 - pc1, m1);
          m0 = fma(a3l0, pl0 - pc0, m0);          m1 = fma(a3l1, pl1 - pc1, m1);
        }
        std2(c.mu + i, m0, m1);
        dot = fma(pc0, m0, dot);
        dot = fma(pc1, m1, dot);
      }
      pl0 = pc0; pl1 = pc1; pc0 = ph0; pc1 = ph1; a3l0 = a3u0; a3l1 = a3u1;
    }
  }
}

__global__ void __launch_bounds__(kThreads, 3) k_fused_pspmv_x2(const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials) {
  __shared__ __align__(16) double sp[2][XTY + 2][XS];
  __shared__ double smem[32];
  __shared__ int s_flag;
  if (ctl->halt) return;                     // unrolled graph body: this pass is over
  const Ctx c = *ctxp;
  if (c.k1_split && ctl->stage == 0) return; // thin stacks: the early stage belongs to k_fused_pspmv_tma
  const int pcur = ctl->pcur;
  const double* p_in = pcur ? c.p2 : c.p;
  double* p_out = pcur ? c.p : c.p2;
  const double beta = ctl->beta, xalpha = ctl->xalpha;
  double acc[1] = {0.0};
  if (ctl->stage == 0) fused_pspmv_x2_body<true>(c, p_in, p_out, beta, xalpha, sp, acc[0]);
  else fused_pspmv_x2_body<false>(c, p_in, p_out, beta, xalpha, sp, acc[0]);
  if (grid_sum_last_block<1>(acc, partials, &ctl->ticket[1], smem, &s_flag) && threadIdx.x == 0) {
    ctl->pcur = pcur ^ 1;
    policy_after_spmv(ctl, acc[0], true, &c);   // Alg. 1 line 7; x += alpha p deferred to the next K1 (or to K2: xnow)
  }
}

}  // namespace cuth
