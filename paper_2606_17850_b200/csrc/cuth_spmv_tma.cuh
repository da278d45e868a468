// cuth_spmv_tma.cuh -- y = A x (cuth_spmv; Alg. 2) with every operand brought in by TMA.
//
// Why: the LDG z-marching SpMV (zmarch_apply_x2) runs the fp64 operator at 0.91 of the measured copy peak but the
// fp32-stored one (27.75 B/row) at only 0.82 at cfg 3 -- more instructions per byte (cvt, predicates) and nothing to hide
// them behind -- the one figure of BASELINE.md below 70 % of the 8 TB/s nominal.  Same cure as K1 (cuth_fused_tma.cuh):
// per plane ONE thread requests boxes of 3-D tensors -- x for the 64 x 8 tile plus its one-cell rim, the three
// off-diagonals (and D0 for the fp64 operator) -- into a ring of four shared-memory stages; completion is an mbarrier
// transaction count; the threads read shared memory only.
//
// A tile is nz + 1 steps: step j waits for plane j (j < nz), takes the thread's own pair of x(j) -- the z + 1 neighbour of
// plane j - 1 -- and forms rows j - 1 of y from the in-plane neighbours and the matrix entries of plane j - 1 (the stage
// before: still resident) and x(j - 2), x(j - 1), D3(j - 2) in registers.  One __syncthreads per step: after it plane
// j - 1's stage is free and is requested again for the plane three ahead.  The planes of ALL tiles of a CTA form one
// stream (persistent over tiles), plane p of the stream living in stage p % 4.
// Cells outside the grid: TMA zero-fills x, and the aligned per-diagonal copies of the matrix have zero tails / stored
// structural zeros, so an absent neighbour is a zero coefficient times a finite value.  Same order of operations per row
// as zmarch_apply_x2: bit-identical y.  Requirements (host): nx % 4 == 0, x 16-byte aligned.
#pragma once
#include "cuth_fused_tma.cuh"

namespace cuth {

constexpr int kSpStages = 4;

template <bool MIXED>
struct SpStage {
  using E = typename std::conditional<MIXED, float, double>::type;
  static constexpr int W1 = K1X + 16 / (int)sizeof(E);  // D1 box: x0 - 16 bytes .. x0+63
  alignas(128) double vx[K1VH][K1VW];                   // x: x0-2 .. x0+65, y0-1 .. y0+8
  alignas(128) E m1[K1Y][W1];
  alignas(128) E m2[K1Y + 1][K1X];                      // rows y0-1 .. y0+7: the entry towards y-1 is the row above's
  alignas(128) E m3[K1Y][K1X];
  alignas(128) double d0[MIXED ? 1 : K1Y][MIXED ? 2 : K1X];   // fp64 operator only (the difference form takes s(z))
  static constexpr uint32_t kBytes = sizeof(double) * K1VH * K1VW + sizeof(E) * (K1Y * W1 + (K1Y + 1) * K1X + K1Y * K1X) +
                                     (MIXED ? 0u : (uint32_t)sizeof(double) * K1Y * K1X);
};
template <bool MIXED>
struct SpSmem {
  SpStage<MIXED> st[kSpStages];
  alignas(8) uint64_t full[kSpStages];
};

template <bool MIXED>
__global__ void __launch_bounds__(kThreads, MIXED ? 4 : 2) k_spmv_tma(DiaDev A, double* __restrict__ y,
    const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmD0, const __grid_constant__ CUtensorMap tm1,
    const __grid_constant__ CUtensorMap tm2, const __grid_constant__ CUtensorMap tm3) {
  extern __shared__ __align__(128) unsigned char sp_smem_raw[];
  using ST = SpStage<MIXED>;
  using E = typename ST::E;
  SpSmem<MIXED>& sm = *reinterpret_cast<SpSmem<MIXED>*>(sp_smem_raw);
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + K1X - 1) / K1X, tiles_y = (nyi + K1Y - 1) / K1Y;
  const int ntiles = tiles_x * tiles_y;
  const int64_t nx = A.nx, np = A.nxny;
  const double* __restrict__ s_layer = A.s_layer;
  const int my_tiles = blockIdx.x < (unsigned)ntiles ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int total_planes = my_tiles * nz;
  constexpr int AL1 = 16 / (int)sizeof(E);
  const int sc0 = 2 + 2 * tx;                          // column of the pair in the x box

  // ---- requests (thread 0): plane rp of this CTA's stream = (tile rk, plane rj), into stage rp % 4
  int rk = 0, rj = 0, rp = 0;
  auto request_next = [&]() {
    const int t = (int)blockIdx.x + rk * (int)gridDim.x;
    const int x0 = (t % tiles_x) * K1X, y0 = (t / tiles_x) * K1Y;
    ST& S = sm.st[rp % kSpStages];
    uint64_t* bar = &sm.full[rp % kSpStages];
    mbar_expect_tx(bar, ST::kBytes);
    tma_load_3d(S.vx, &tmX, bar, x0 - 2, y0 - 1, rj);
    tma_load_3d(S.m1, &tm1, bar, x0 - AL1, y0, rj);
    tma_load_3d(S.m2, &tm2, bar, x0, y0 - 1, rj);
    tma_load_3d(S.m3, &tm3, bar, x0, y0, rj);
    if (!MIXED) tma_load_3d(S.d0, &tmD0, bar, x0, y0, rj);
    if (++rj == nz) { rj = 0; ++rk; }
    ++rp;
  };
  if (tid == 0) {
    for (int s = 0; s < kSpStages; ++s) mbar_init(&sm.full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int s = 0; s < kSpStages && s < total_planes; ++s) request_next();
  }
  __syncthreads();

  int pl = 0;                                          // planes of the stream consumed so far
  for (int k = 0; k < my_tiles; ++k) {
    const int t = (int)blockIdx.x + k * (int)gridDim.x;
    const int x = (t % tiles_x) * K1X + 2 * tx, yy = (t / tiles_x) * K1Y + ty;
    const bool own = x < nxi && yy < nyi;              // nx even: x + 1 < nx too
    const int64_t col = own ? x + nx * (int64_t)yy : 0;
    double2 v_lo = make_double2(0.0, 0.0), v_c = v_lo;
    double a3l0 = 0.0, a3l1 = 0.0;
    int prev = 0;
    for (int j = 0; j <= nz; ++j) {
      // ---- 1. plane j: the thread's own pair
      double2 v_hi = MIXED ? v_c : make_double2(0.0, 0.0);
      int cur = prev;
      if (j < nz) {
        cur = pl % kSpStages;
        mbar_wait(&sm.full[cur], (uint32_t)((pl / kSpStages) & 1));
        v_hi = *reinterpret_cast<const double2*>(&sm.st[cur].vx[ty + 1][sc0]);
      }
      // ---- 2. rows of plane j - 1
      if (j >= 1) {
        const ST& S = sm.st[prev];
        const double vl = S.vx[ty + 1][sc0 - 1], vr = S.vx[ty + 1][sc0 + 2];
        const double2 v2l = *reinterpret_cast<const double2*>(&S.vx[ty][sc0]);
        const double2 v2u = *reinterpret_cast<const double2*>(&S.vx[ty + 2][sc0]);
        const double2 a1 = k1_ld_pair<MIXED>(&S.m1[ty][AL1 + 2 * tx]);
        const double a1l = (double)S.m1[ty][AL1 + 2 * tx - 1];
        const double2 a2u = k1_ld_pair<MIXED>(&S.m2[ty + 1][2 * tx]);
        const double2 a2l = k1_ld_pair<MIXED>(&S.m2[ty][2 * tx]);
        const double2 a3u = k1_ld_pair<MIXED>(&S.m3[ty][2 * tx]);
        double y0, y1;
        if (!MIXED) {
          const double2 d0 = *reinterpret_cast<const double2*>(&S.d0[MIXED ? 0 : ty][MIXED ? 0 : 2 * tx]);
          y0 = d0.x * v_c.x;              y1 = d0.y * v_c.y;
          y0 = fma(a1.x, v_c.y, y0);      y1 = fma(a1.x, v_c.x, y1);
          y0 = fma(a1l, vl, y0);          y1 = fma(a1.y, vr, y1);
          y0 = fma(a2u.x, v2u.x, y0);     y1 = fma(a2u.y, v2u.y, y1);
          y0 = fma(a2l.x, v2l.x, y0);     y1 = fma(a2l.y, v2l.y, y1);
          y0 = fma(a3u.x, v_hi.x, y0);    y1 = fma(a3u.y, v_hi.y, y1);
          y0 = fma(a3l0, v_lo.x, y0);     y1 = fma(a3l1, v_lo.y, y1);
        } else {
          const double s = s_layer[j - 1];
          const double2 lo = j > 1 ? v_lo : v_c;
          y0 = s * v_c.x;                         y1 = s * v_c.y;
          y0 = fma(a1.x, v_c.y - v_c.x, y0);      y1 = fma(a1.x, v_c.x - v_c.y, y1);
          y0 = fma(a1l, vl - v_c.x, y0);          y1 = fma(a1.y, vr - v_c.y, y1);
          y0 = fma(a2u.x, v2u.x - v_c.x, y0);     y1 = fma(a2u.y, v2u.y - v_c.y, y1);
          y0 = fma(a2l.x, v2l.x - v_c.x, y0);     y1 = fma(a2l.y, v2l.y - v_c.y, y1);
          y0 = fma(a3u.x, v_hi.x - v_c.x, y0);    y1 = fma(a3u.y, v_hi.y - v_c.y, y1);
          y0 = fma(a3l0, lo.x - v_c.x, y0);       y1 = fma(a3l1, lo.y - v_c.y, y1);
        }
        if (own) std2(y + col + (int64_t)(j - 1) * np, y0, y1);
        a3l0 = a3u.x; a3l1 = a3u.y;
      }
      // ---- 3. plane j - 1's stage is consumed: ask for the plane three ahead into it
      __syncthreads();
      if (j >= 1 && tid == 0 && rp < total_planes) request_next();
      v_lo = v_c; v_c = v_hi;
      if (j < nz) { prev = cur; ++pl; }
    }
  }
}

}  // namespace cuth
