// cuth_cheb_pair.cuh -- TWO consecutive passes of the Chebyshev apply in one kernel (fp32 modes).
//
// The polynomial preconditioner has no reduction between its SpMVs, so nothing forces a
// grid-wide barrier between pass i and pass i+1:
//
//   W = U + c1_i     (U - V) + c2_i     (r - A U)        U = Z_{i+1}, V = Z_i, W = Z_{i+2}
//   Y = W + c1_{i+1} (W - U) + c2_{i+1} (r - A W)        Y = Z_{i+3}
//
// A CTA owns a region of QX x QY columns of the x-y plane and marches in z, a thread owns two x-adjacent
// columns (as in k_cheb_mid_f32x2, whose row arithmetic this repeats term for term).  Every thread forms W
// for its pair on plane k from U read through L1/L2 exactly like the single pass; the plane of W goes to
// shared memory; the threads that are not on the rim of the region then form Y on plane k-1 from the
// shared W plane (in-plane neighbours) and their own registers (W on planes k-2, k-1, k; the matrix row, r
// and U of plane k-1, kept from the step before).  W never makes the HBM round trip as a stencil input, the
// matrix row and r are fetched once for two passes: a row moves  M + 5 * 4 B  (U, V, r read; W, Y written)
// instead of 2 (M + 16).  The rim (one pair left and right, one row above and below) is recomputed by the
// neighbouring CTA: 360 of 512 cells of a region are interior (QY = 8), their operands are L2 hits.
// One barrier per plane: W(k) is computed before it and stored after it, Y(k-1) reads the plane stored one
// step earlier, so a buffer of the two-plane ring is never written while still read.  The x-neighbours of a
// pair (U for W, W for Y, and the D1 entry to the left) come from the adjacent lanes by warp shuffle: a warp
// is one row of the region, and what lanes 0 / 31 cannot get that way only feeds the outer cell of a rim pair,
// which nobody reads.  The first and the last plane (where the band leaves [0, N)) are peeled, so the planes
// in between run without bounds predicates.
// Outputs go to the two buffers that are not inputs (neighbouring CTAs still read U and V), see cheb_schedule.
#pragma once
#include "cuth_cheb.cuh"

namespace cuth {

constexpr int QX = 64, QY = 8;                         // region: 32 column pairs x 8 rows = one thread each
constexpr int QIX = QX - 4, QIY = QY - 2;              // interior written by this CTA: 60 x 6 columns
static_assert(QX / 2 * QY == kThreads, "one thread per column pair of the region");

template <class M>
__global__ void __launch_bounds__(kThreads, 4) k_cheb_pair_f32(const Ctx* __restrict__ ctxp, int step, int old, int cur,
                                                             int wout, int yout) {
  __shared__ __align__(8) float sW[2][QY][QX];
  const Ctx c = *ctxp;
  const DiaDev& A = c.A;
  const float c1a = (float)ctxp->cheb_c1[step], c2a = (float)ctxp->cheb_c2[step];
  const float c1b = (float)ctxp->cheb_c1[step + 1], c2b = (float)ctxp->cheb_c2[step + 1];
  const float* __restrict__ U = (const float*)ctxp->cd[cur];
  const float* __restrict__ V = (const float*)ctxp->cd[old];
  float* __restrict__ Wg = (float*)ctxp->cd[wout];
  float* __restrict__ Yg = (float*)ctxp->cd[yout];
  const float* __restrict__ r32 = (const float*)c.crc;
  // the pointers come out of a struct in memory: tell the compiler they are global (LDG / STG, not generic)
  __builtin_assume(__isGlobal(U)); __builtin_assume(__isGlobal(V)); __builtin_assume(__isGlobal(Wg));
  __builtin_assume(__isGlobal(Yg)); __builtin_assume(__isGlobal(r32));
  __builtin_assume(__isGlobal(M::d1(A))); __builtin_assume(__isGlobal(M::d2(A))); __builtin_assume(__isGlobal(M::d3(A)));
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + QIX - 1) / QIX, tiles_y = (nyi + QIY - 1) / QIY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t nx = A.nx, np = A.nxny;
  // U, V, r and the matrix are only read by this kernel: non-coherent loads
  auto ld2 = [](const float* p) { return __ldg(reinterpret_cast<const float2*>(p)); };
  const float ms = M::inv(A);
  const float2 z2 = make_float2(0.f, 0.f);
  const bool rim = tx == 0 || tx == 31 || ty == 0 || ty == QY - 1;
  constexpr unsigned kAll = 0xffffffffu;

  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x = bx * QIX - 2 + 2 * tx, y = by * QIY - 1 + ty;        // x even; nx even: x + 1 < nx with x
    const bool live = x >= 0 && x < nxi && y >= 0 && y < nyi;
    const bool inner = live && !rim;
    const int64_t c0 = live ? x + nx * (int64_t)y : 0;

    // one pointer per stream, bumped by a plane per step (no per-load index arithmetic)
    const float* pU = U + c0; const float* pV = V + c0; const float* pR = r32 + c0;
    const typename M::elem* q1 = M::d1(A) + c0; const typename M::elem* q2 = M::d2(A) + c0;
    const typename M::elem* q3 = M::d3(A) + c0;
    float* pW = Wg + c0; float* pY = Yg + c0 - np;                       // Y trails W by a plane
    const bool row0 = y == 0, rowN = y == nyi - 1, cellN = c0 + 2 == np;

    float2 u_lo = z2, u_c = live ? ld2(pU) : z2;                        // U on planes k-1, k
    float2 w_lo = z2, w_c = z2;                                         // W on planes k-2, k-1
    float2 a3l_w = z2, a3l_y = z2;                                      // D3 below plane k / below plane k-1
    // row of plane k-1, kept for Y
    float pf1l = 0.f, pf1a = 0.f, pf1b = 0.f, ps = 0.f;
    float2 pf2u = z2, pf2l = z2, pa3u = z2, pr = z2;

    // One step: W on plane k (if HAS_W), barrier, Y on plane k-1 (if HAS_Y).  FIRST / LAST: plane 0 / nz-1,
    // the only ones where a +-nx, +-1 or +nx*ny neighbour of a live cell can fall outside [0, N).
    auto do_step = [&](auto first_t, auto last_t, auto has_w_t, auto has_y_t, int k) {
      constexpr bool FIRST = decltype(first_t)::value, LAST = decltype(last_t)::value;
      constexpr bool HAS_W = decltype(has_w_t)::value, HAS_Y = decltype(has_y_t)::value;
      float2 w = z2, u_hi = z2, rv = z2, f2u = z2, f2l = z2, a3u = z2;
      float f1l = 0.f, f1a = 0.f, f1b = 0.f, s = 0.f;
      if (HAS_W) {
        // x-neighbours of the pair and the D1 entry to its left: from the adjacent lanes
        const float vl = __shfl_up_sync(kAll, u_c.y, 1), vr = __shfl_down_sync(kAll, u_c.x, 1);
        // every global load of the step first, back to back; the shuffle that depends on one of them after
        float2 f1p = z2, v2u = z2, v2l = z2, zo = z2;
        if (live) {
          const bool up1 = !LAST || !cellN, up2 = !LAST || !rowN, lo2 = !FIRST || !row0;
          f1p = up1 ? M::ldp(q1, ms) : make_float2(M::ld(q1, ms), 0.f);
          f2u = up2 ? M::ldp(q2, ms) : z2; f2l = lo2 ? M::ldp(q2 - nx, ms) : z2;
          if (!LAST) { a3u = M::ldp(q3, ms); u_hi = ld2(pU + np); } else { u_hi = u_c; }
          v2u = up2 ? ld2(pU + nx) : u_c; v2l = lo2 ? ld2(pU - nx) : u_c;
          rv = ld2(pR);
          zo = ld2(pV);
        }
        f1a = f1p.x; f1b = f1p.y;
        f1l = __shfl_up_sync(kAll, f1b, 1);
        if (live) {
          s = (float)A.s_layer[k];
          float a0 = s * u_c.x, a1 = s * u_c.y;
          a0 += f1a * (u_c.y - u_c.x);     a1 += f1a * (u_c.x - u_c.y);
          a0 += f1l * (vl - u_c.x);        a1 += f1b * (vr - u_c.y);
          a0 += f2u.x * (v2u.x - u_c.x);   a1 += f2u.y * (v2u.y - u_c.y);
          a0 += f2l.x * (v2l.x - u_c.x);   a1 += f2l.y * (v2l.y - u_c.y);
          a0 += a3u.x * (u_hi.x - u_c.x);  a1 += a3u.y * (u_hi.y - u_c.y);
          a0 += a3l_w.x * (u_lo.x - u_c.x); a1 += a3l_w.y * (u_lo.y - u_c.y);
          w = make_float2(u_c.x + c1a * (u_c.x - zo.x) + c2a * (rv.x - a0),
                          u_c.y + c1a * (u_c.y - zo.y) + c2a * (rv.y - a1));
          if (inner) *reinterpret_cast<float2*>(pW) = w;
        }
      }
      __syncthreads();                                   // plane k-1 of W is complete; plane k-2 no longer read
      if (HAS_W) *reinterpret_cast<float2*>(&sW[k & 1][ty][2 * tx]) = w;
      if (HAS_Y) {
        const float wl = __shfl_up_sync(kAll, w_c.y, 1), wr = __shfl_down_sync(kAll, w_c.x, 1);
        if (inner) {
          const float (*P)[QX] = sW[(k - 1) & 1];
          const float2 wu = *reinterpret_cast<const float2*>(&P[ty + 1][2 * tx]);
          const float2 wd = *reinterpret_cast<const float2*>(&P[ty - 1][2 * tx]);
          float a0 = ps * w_c.x, a1 = ps * w_c.y;
          a0 += pf1a * (w_c.y - w_c.x);    a1 += pf1a * (w_c.x - w_c.y);
          a0 += pf1l * (wl - w_c.x);       a1 += pf1b * (wr - w_c.y);
          a0 += pf2u.x * (wu.x - w_c.x);   a1 += pf2u.y * (wu.y - w_c.y);
          a0 += pf2l.x * (wd.x - w_c.x);   a1 += pf2l.y * (wd.y - w_c.y);
          a0 += pa3u.x * (w.x - w_c.x);    a1 += pa3u.y * (w.y - w_c.y);     // pa3u = 0 on the top plane
          a0 += a3l_y.x * (w_lo.x - w_c.x); a1 += a3l_y.y * (w_lo.y - w_c.y);
          *reinterpret_cast<float2*>(pY) = make_float2(w_c.x + c1b * (w_c.x - u_lo.x) + c2b * (pr.x - a0),
                                                       w_c.y + c1b * (w_c.y - u_lo.y) + c2b * (pr.y - a1));
        }
      }
      // ---- rotate: plane k becomes plane k-1
      a3l_y = pa3u;
      pf1l = f1l; pf1a = f1a; pf1b = f1b; ps = s; pf2u = f2u; pf2l = f2l; pa3u = a3u; pr = rv;
      w_lo = w_c; w_c = w;
      a3l_w = a3u;
      u_lo = u_c; u_c = u_hi;
      pU += np; pV += np; pR += np; q1 += np; q2 += np; q3 += np; pW += np; pY += np;
    };
    constexpr std::true_type T{};
    constexpr std::false_type F{};

    __syncthreads();                                                    // previous tile done with sW
    do_step(T, F, T, F, 0);                                             // nz >= 2: plane 0 is not the last
#pragma unroll 2
    for (int k = 1; k < nz - 1; ++k) do_step(F, F, T, T, k);
    do_step(F, T, T, T, nz - 1);
    do_step(F, F, F, T, nz);
  }
}

}  // namespace cuth
