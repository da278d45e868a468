// cuth_cheb_pair.cuh -- TWO consecutive passes of the Chebyshev apply in one kernel (fp32 mode).
//
// The polynomial preconditioner has no reduction between its SpMVs, so nothing forces a
// grid-wide barrier between pass i and pass i+1: a CTA can compute W = Z_{i+2} on its tile plus a one-cell
// in-plane ring (from U = Z_{i+1} on a two-cell ring), and then Y = Z_{i+3} on the tile, without W ever
// leaving the SM.  Per two passes a row then moves  M + 5 * 4 B  (matrix once; U, V = Z_i, r read; W, Y
// written) instead of 2 * (M + 16): 31.75 instead of 55.5 B/row on A2.  The ring is recomputed by the
// neighbouring CTA as part of its own tile (same arithmetic, same order, hence the same bits).
//
//   W = U + c1_i     (U - V) + c2_i     (r - A U)        on (TX+2) x (TY+2), planes z-1 .. z+1 kept in smem
//   Y = W + c1_{i+1} (W - U) + c2_{i+1} (r - A W)        on  TX    x  TY
//
// A CTA marches in z; per plane: (1) stage plane z+2 of U (tile + 2-ring) in shared memory, (2) W(z+1) on the
// tile + 1-ring from the three staged U planes, (3) Y(z) on the tile from the three staged W planes.  Rings of 4
// planes for U and W make two barriers per plane enough.  Outputs go to the two buffers that are NOT inputs
// (neighbouring CTAs still read U, V of this tile), see cheb_schedule.
#pragma once
#include "cuth_cheb.cuh"

namespace cuth {

constexpr int PTX = 64, PTY = 8;                       // interior tile (columns)
constexpr int PWX = PTX + 2, PWY = PTY + 2;            // W region: 1-ring
constexpr int PUX = PTX + 4, PUY = PTY + 4;            // U region: 2-ring
constexpr int kPairWCells = PWX * PWY;                 // 660
constexpr int kPairUCells = PUX * PUY;                 // 816
constexpr int kPairWPerThread = (kPairWCells + kThreads - 1) / kThreads;   // 3
constexpr int kPairICells = PTX * PTY;                 // 512
constexpr int kPairIPerThread = kPairICells / kThreads;                    // 2

template <class M>
__global__ void __launch_bounds__(kThreads, 3) k_cheb_pair_f32(const Ctx* __restrict__ ctxp, int step, int old, int cur,
                                                             int wout, int yout) {
  __shared__ float sU[4][PUY][PUX];
  __shared__ float sW[4][PWY][PWX];
  const Ctx c = *ctxp;
  const DiaDev& A = c.A;
  const float c1a = (float)ctxp->cheb_c1[step], c2a = (float)ctxp->cheb_c2[step];
  const float c1b = (float)ctxp->cheb_c1[step + 1], c2b = (float)ctxp->cheb_c2[step + 1];
  const float* __restrict__ U = (const float*)ctxp->cd[cur];
  const float* __restrict__ V = (const float*)ctxp->cd[old];
  float* __restrict__ Wg = (float*)ctxp->cd[wout];
  float* __restrict__ Yg = (float*)ctxp->cd[yout];
  const float* __restrict__ r32 = (const float*)c.crc;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + PTX - 1) / PTX, tiles_y = (nyi + PTY - 1) / PTY;
  const int ntiles = tiles_x * tiles_y;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const float ms = M::inv(A);
  const int tid = threadIdx.x;

  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x0 = bx * PTX, y0 = by * PTY;

    // stage one plane of U (tile + 2-ring) into ring slot zz & 3; planes / cells outside the grid are 0
    auto stage_U = [&](int zz) {
      float (*dst)[PUX] = sU[zz & 3];
      const bool zin = zz >= 0 && zz < nz;
      for (int q = tid; q < kPairUCells; q += kThreads) {
        const int uy = q / PUX, ux = q - uy * PUX;
        const int gx = x0 - 2 + ux, gy = y0 - 2 + uy;
        float v = 0.f;
        if (zin && gx >= 0 && gx < nxi && gy >= 0 && gy < nyi) v = U[gx + nx * (int64_t)gy + (int64_t)zz * np];
        dst[uy][ux] = v;
      }
    };
    // W on the tile + 1-ring for plane zz (needs U planes zz-1, zz, zz+1 staged); written to smem and, on the tile, to HBM
    float a3l_w[kPairWPerThread];
#pragma unroll
    for (int k = 0; k < kPairWPerThread; ++k) a3l_w[k] = 0.f;
    auto compute_W = [&](int zz) {
      float (*dst)[PWX] = sW[zz & 3];
      const bool zin = zz >= 0 && zz < nz;
      const float s = zin ? (float)A.s_layer[zz] : 0.f;
      float (*Uc)[PUX] = sU[zz & 3];
      float (*Ul)[PUX] = sU[(zz + 3) & 3];
      float (*Uh)[PUX] = sU[(zz + 1) & 3];
#pragma unroll
      for (int k = 0; k < kPairWPerThread; ++k) {
        const int q = tid + k * kThreads;
        if (q >= kPairWCells) break;
        const int wy = q / PWX, wx = q - wy * PWX;
        const int gx = x0 - 1 + wx, gy = y0 - 1 + wy;
        float w = 0.f;
        if (zin && gx >= 0 && gx < nxi && gy >= 0 && gy < nyi) {
          const int64_t i = gx + nx * (int64_t)gy + (int64_t)zz * np;
          const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = zz + 1 < nz;
          const float a1u = up1 ? M::e1(A, i, ms) : 0.f, a1l = lo1 ? M::e1(A, i - 1, ms) : 0.f;
          const float a2u = up2 ? M::e2(A, i, ms) : 0.f, a2l = lo2 ? M::e2(A, i - nx, ms) : 0.f;
          const float a3u = up3 ? M::e3(A, i, ms) : 0.f;
          const float vi = V[i], ri = r32[i];
          const int ux = wx + 1, uy = wy + 1;                    // same cell in the U region
          const float u = Uc[uy][ux];
          float au = s * u;
          au += a1u * (Uc[uy][ux + 1] - u); au += a1l * (Uc[uy][ux - 1] - u);
          au += a2u * (Uc[uy + 1][ux] - u); au += a2l * (Uc[uy - 1][ux] - u);
          au += a3u * (Uh[uy][ux] - u);     au += a3l_w[k] * (Ul[uy][ux] - u);
          w = u + c1a * (u - vi) + c2a * (ri - au);
          a3l_w[k] = a3u;
          if (wx >= 1 && wx <= PTX && wy >= 1 && wy <= PTY) Wg[i] = w;      // the tile itself
        }
        dst[wy][wx] = w;
      }
    };

    __syncthreads();                                   // previous tile done with the rings
    stage_U(-1); stage_U(0); stage_U(1);
    // W(-1) = 0
    for (int q = tid; q < kPairWCells; q += kThreads) sW[3][q / PWX][q % PWX] = 0.f;
    __syncthreads();
    compute_W(0);
    float a3l_y[kPairIPerThread];
#pragma unroll
    for (int k = 0; k < kPairIPerThread; ++k) a3l_y[k] = 0.f;

    for (int z = 0; z < nz; ++z) {
      stage_U(z + 2);
      __syncthreads();                                 // U(z+2) staged; W(z) complete
      compute_W(z + 1);
      __syncthreads();                                 // W(z+1) complete
      // ---- Y(z) on the tile
      const float s = (float)A.s_layer[z];
      float (*Wc)[PWX] = sW[z & 3];
      float (*Wl)[PWX] = sW[(z + 3) & 3];
      float (*Wh)[PWX] = sW[(z + 1) & 3];
      float (*Uc)[PUX] = sU[z & 3];
#pragma unroll
      for (int k = 0; k < kPairIPerThread; ++k) {
        const int q = tid + k * kThreads;
        const int iy = q / PTX, ix = q - iy * PTX;
        const int gx = x0 + ix, gy = y0 + iy;
        if (gx < nxi && gy < nyi) {
          const int64_t i = gx + nx * (int64_t)gy + (int64_t)z * np;
          const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = z + 1 < nz;
          const float a1u = up1 ? M::e1(A, i, ms) : 0.f, a1l = lo1 ? M::e1(A, i - 1, ms) : 0.f;
          const float a2u = up2 ? M::e2(A, i, ms) : 0.f, a2l = lo2 ? M::e2(A, i - nx, ms) : 0.f;
          const float a3u = up3 ? M::e3(A, i, ms) : 0.f;
          const float ri = r32[i];
          const int wx = ix + 1, wy = iy + 1;
          const float w = Wc[wy][wx], u = Uc[iy + 2][ix + 2];
          float aw = s * w;
          aw += a1u * (Wc[wy][wx + 1] - w); aw += a1l * (Wc[wy][wx - 1] - w);
          aw += a2u * (Wc[wy + 1][wx] - w); aw += a2l * (Wc[wy - 1][wx] - w);
          aw += a3u * (Wh[wy][wx] - w);     aw += a3l_y[k] * (Wl[wy][wx] - w);
          Yg[i] = w + c1b * (w - u) + c2b * (ri - aw);
          a3l_y[k] = a3u;
        }
      }
    }
  }
}

}  // namespace cuth
