// cuth_fused_tma.cuh -- K1 (k_fused_pspmv_x2: p' = M^-1 r + beta p, x += alpha_prev p, mu = A p', p'.mu; see
// cuth_fused.cuh / cuth_fused_x2.cuh) with its streamed operands brought in by TMA.
//
// Why: both LDG versions of K1 take ~0.22-0.24 ms at cfg-3 size whatever the matrix bytes (fp64 operator 79.5 B/row,
// fp32-stored 67.75 B/row): they are bound by the load instructions a thread can keep in flight at 3 CTAs/SM, not by
// HBM (ncu: long-scoreboard stalls, issue slots ~35 % busy).  Here no register holds a byte in flight:
// per plane, ONE thread requests boxes of 3-D tensors (x, y, z) with cp.async.bulk.tensor -- r, p and the diagonal
// (1/D0, or D0 itself in fp64 mode) for the tile plus its one-cell rim, and the three off-diagonals -- three steps
// ahead into a ring of shared-memory stages; completion is an mbarrier transaction count.
//
// Structure of a tile (TX x TY = 64 x 8 columns, 256 threads, a thread owns two x-adjacent columns and marches in z):
// nz + 1 steps, step j forms plane j of p' (own pair + the thread's share of the 144 rim cells, from the staged
// r, p, D) and row-plane j - 1 of mu (matrix entries of plane j - 1 from the stage, p' of planes j-2, j-1, j from
// registers and from the two-plane shared ring).  All operands of a step are read from the stage into registers
// BEFORE the step's one __syncthreads, so that the same barrier that orders the p' ring frees the stage for the plane
// three steps ahead (no "empty" mbarriers).  The steps of ALL tiles of a CTA form one stream: the ring keeps running
// across tile boundaries, the pipeline is filled once per kernel, not once per tile.
//
// Cells outside the grid: TMA zero-fills them, and the aligned per-diagonal copies of the matrix have zero tails, so
// an absent neighbour is a zero coefficient times a finite value; p' of rim / ragged cells outside the grid is forced
// to 0 (1/D0 is not finite there).  x is the caller's buffer (its address is not known when the graph is built):
// plain 16-byte loads, prefetched one plane ahead; p', x, mu leave through plain 16-byte stores.
// Requirements (checked on the host): nx % 4 == 0 (tensor-map strides are multiples of 16 bytes), Jacobi or no
// preconditioner (with Chebyshev z is a separate vector and K1 is a small part of the iteration).
#pragma once
#include "cuth_cheb_pair_tma.cuh"
#include "cuth_fused_x2.cuh"

namespace cuth {

constexpr int kK1Stages = 3;
// Split-phase synchronisation of the p' ring (compile-time option, OFF: measured on B200 it changes nothing -- cfg 3 MIXED
// 1.347 vs 1.354 s, cfg 3 FP64 1.376 vs 1.369 s, cfg 4 FP64 24.44 vs 24.26 s, cfg 5 2.299 vs 2.311 s for 40 steps; K1 fp32-stored
// 0.187 vs 0.190 ms -- so the per-step barrier is not what bounds the kernel, and the simpler form is kept).  A step's only CTA-wide dependency is "plane j of p' is complete
// before the NEXT step reads its in-plane neighbours"; with __syncthreads every warp waits for the slowest one in every
// step (ncu, round 2: stalled_barrier 4.9 warps per issue at 2 CTAs/SM).  Instead each warp ARRIVES on an mbarrier
// right after writing its part of plane j and WAITS for that phase only one step later, just before writing plane j + 1:
// warps may drift a step apart.  The wait of phase s - 1 also tells thread 0 that every warp has read the operands of step
// s - 1 out of its stage, so that stage can be requested again (for step s + 2).  Three ring planes make it safe: plane
// (s - 1) % 3 is read by the mu rows of step s and overwritten in step s + 2, whose writers have passed the wait of phase
// s + 1, i.e. every warp has finished step s.  0 = one __syncthreads per step.
#ifndef CUTH_K1_SPLIT
#define CUTH_K1_SPLIT 0
#endif
constexpr int kK1Ring = CUTH_K1_SPLIT ? 3 : 2;
__device__ __forceinline__ void mbar_arrive(uint64_t* b) {
  asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
constexpr int K1X = XTX, K1Y = XTY;                      // 64 x 8 columns per tile (as k_fused_pspmv_x2)
constexpr int K1VW = K1X + 4;                            // vector box: x0-2 .. x0+65 (16-byte aligned start, one-cell rim)
constexpr int K1VH = K1Y + 2;                            // rows y0-1 .. y0+TY

// One stage = the vectors of plane j and the matrix of plane j - 1.  Every member starts on a 128-byte boundary.
template <bool MIXED>
struct K1Stage {
  using E = typename std::conditional<MIXED, float, double>::type;
  static constexpr int W1 = K1X + 16 / (int)sizeof(E);  // D1 box: x0 - 16 bytes .. x0+63 (the entry towards x-1 is the left one's)
  alignas(128) double vz[K1VH][K1VW];                   // r
  alignas(128) double vp[K1VH][K1VW];                   // p (old direction)
  // the diagonal operand: fp32(1/D0) with the fp32-stored operator (box starts at x0 - 4 floats = 16 bytes: four more
  // columns), D0 itself with the fp64 operator
  using VD = typename std::conditional<MIXED, float, double>::type;
  static constexpr int VDW = MIXED ? K1VW + 4 : K1VW, VDX = MIXED ? 4 : 2;   // box width; elements in front of the tile
  alignas(128) VD vd[K1VH][VDW];
  alignas(128) E m1[K1Y][W1];
  alignas(128) E m2[K1Y + 1][K1X];                      // rows y0-1 .. y0+TY-1: the entry towards y-1 is the row above's
  alignas(128) E m3[K1Y][K1X];
  static constexpr uint32_t kVecBytes = 2u * sizeof(double) * K1VH * K1VW + sizeof(VD) * K1VH * VDW;
  static constexpr uint32_t kMatBytes = sizeof(E) * (K1Y * W1 + (K1Y + 1) * K1X + K1Y * K1X);
};
template <bool MIXED>
struct K1Smem {
  K1Stage<MIXED> st[kK1Stages];
  alignas(16) double sp[kK1Ring][K1VH][XS];             // p' ring: (tile + rim) planes of the last kK1Ring steps
  alignas(8) uint64_t full[kK1Stages];
  alignas(8) uint64_t ringbar;                          // split-phase CTA barrier of the p' ring: one arrival per warp and step
  double red[32];
  int s_flag;
};

struct K1Maps { CUtensorMap z, p, p2, d, m1, m2, m3; };

template <bool MIXED>
__device__ __forceinline__ double2 k1_ld_pair(const typename K1Stage<MIXED>::E* q) {
  if (MIXED) { const float2 f = *reinterpret_cast<const float2*>(q); return make_double2((double)f.x, (double)f.y); }
  else return *reinterpret_cast<const double2*>(q);
}

template <bool MIXED>
__device__ __forceinline__ void fused_pspmv_tma_body(const Ctx& c, K1Smem<MIXED>& sm, double* __restrict__ p_out,
                                                     const double beta, const double xalpha, const CUtensorMap* tmZ,
                                                     const CUtensorMap* tmP, const CUtensorMap* tmD,
                                                     const CUtensorMap* tm1, const CUtensorMap* tm2,
                                                     const CUtensorMap* tm3, double& dot) {
  using ST = K1Stage<MIXED>;
  using E = typename ST::E;
  const DiaDev& A = c.A;
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + K1X - 1) / K1X, tiles_y = (nyi + K1Y - 1) / K1Y;
  const int ntiles = tiles_x * tiles_y;
  const int64_t nx = A.nx, np = A.nxny;
  const bool jac = c.jacobi != 0;
  double* __restrict__ xg = c.x;
  double* __restrict__ mug = c.mu;
  const double* __restrict__ s_layer = A.s_layer;
  __builtin_assume(__isGlobal(xg)); __builtin_assume(__isGlobal(mug)); __builtin_assume(__isGlobal(p_out));
  const int my_tiles = blockIdx.x < (unsigned)ntiles ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int spt = nz + 1;                              // steps per tile
  const int total = my_tiles * spt;
  constexpr int AL1 = 16 / (int)sizeof(E);             // elements of the 16 bytes in front of the D1 box
  const int sc0 = 2 + 2 * tx;                          // column of the pair in the p' ring and in the vector boxes

  // ---- requests (thread 0): step r of this CTA's stream = (tile rk, plane rj)
  int rk = 0, rj = 0, rslot = 0;
  auto request_next = [&]() {
    const int t = (int)blockIdx.x + rk * (int)gridDim.x;
    const int x0 = (t % tiles_x) * K1X, y0 = (t / tiles_x) * K1Y;
    ST& S = sm.st[rslot];
    uint64_t* bar = &sm.full[rslot];
    mbar_expect_tx(bar, (rj < nz ? ST::kVecBytes : 0u) + (rj >= 1 ? ST::kMatBytes : 0u));
    if (rj < nz) {
      tma_load_3d(S.vz, tmZ, bar, x0 - 2, y0 - 1, rj);
      tma_load_3d(S.vp, tmP, bar, x0 - 2, y0 - 1, rj);
      tma_load_3d(S.vd, tmD, bar, x0 - ST::VDX, y0 - 1, rj);
    }
    if (rj >= 1) {
      tma_load_3d(S.m1, tm1, bar, x0 - AL1, y0, rj - 1);
      tma_load_3d(S.m2, tm2, bar, x0, y0 - 1, rj - 1);
      tma_load_3d(S.m3, tm3, bar, x0, y0, rj - 1);
    }
    if (++rj == spt) { rj = 0; ++rk; }
    if (++rslot == kK1Stages) rslot = 0;
  };
  if (tid == 0) {
    for (int s = 0; s < kK1Stages; ++s) mbar_init(&sm.full[s], 1);
    mbar_init(&sm.ringbar, kThreads / 32);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    for (int s = 0; s < kK1Stages && s < total; ++s) request_next();
  }
  __syncthreads();

  // ---- per-tile state
  int x = 0, y = 0;
  bool own = false, halo_role = false, halo_in = false;
  int64_t col = 0;
  int hr = 0, hc = 0, hbr = 0, hbc = 0;                // rim cell: place in the p' ring / in the vector boxes
  double pc0 = 0.0, pc1 = 0.0, pl0 = 0.0, pl1 = 0.0, a3l0 = 0.0, a3l1 = 0.0;
  double2 dcur = make_double2(0.0, 0.0);               // fp64 operator: D0 of the plane mu is formed for
  // x is the caller's buffer (no tensor map): plain loads, issued TWO p'-planes ahead -- across tile boundaries too, so that
  // no step ever waits for HBM (round 2a loaded plane 0 of every tile synchronously: ~1 us of the ~17 us of a tile)
  double2 xq0 = make_double2(0.0, 0.0), xq1 = xq0;     // x of the plane of this step / of the next p'-step
  auto tile_col = [&](int kk, bool* o) -> int64_t {    // first row of this thread's pair in tile kk; *o: inside the grid
    const int t = (int)blockIdx.x + kk * (int)gridDim.x;
    const int xx = (t % tiles_x) * K1X + 2 * tx, yy = (t / tiles_x) * K1Y + ty;
    *o = xx < nxi && yy < nyi;
    return *o ? xx + nx * (int64_t)yy : 0;
  };
  const bool do_x = xalpha != 0.0;                     // nothing pending (first iteration, or K2 / k_flush_x applied it): x untouched
  if (my_tiles > 0 && do_x) {
    bool on; const int64_t c0 = tile_col(0, &on);
    if (on) { xq0 = ldd2(xg + c0); xq1 = ldd2(xg + c0 + np); }       // nz >= 2
  }
  uint32_t ph = 0;                                     // bit S: parity of the next fill of stage S
  int slot = 0, j = 0, k = 0;
  int rw = 0, rr = kK1Ring - 1;                        // ring plane written in this step / written in the step before

  for (int s = 0; s < total; ++s) {
    if (j == 0) {                                      // a new tile
      const int t = (int)blockIdx.x + k * (int)gridDim.x;
      const int bx = t % tiles_x, by = t / tiles_x;
      x = bx * K1X + 2 * tx; y = by * K1Y + ty;
      own = x < nxi && y < nyi;                        // nx even: x + 1 < nx too
      col = own ? x + nx * (int64_t)y : 0;
      const int h = tx < kHaloX2PerWarp ? ty * kHaloX2PerWarp + tx : kHaloX2;
      int hx = -1, hy = -1;
      if (h < K1X)                { hx = bx * K1X + h;          hy = by * K1Y - 1;   hr = 0;        hc = 2 + h; }
      else if (h < 2 * K1X)       { hx = bx * K1X + (h - K1X);  hy = by * K1Y + K1Y; hr = K1Y + 1;  hc = 2 + h - K1X; }
      else if (h < 2 * K1X + K1Y) { hx = bx * K1X - 1;          hy = by * K1Y + (h - 2 * K1X);       hr = h - 2 * K1X + 1;       hc = 1; }
      else if (h < kHaloX2)       { hx = bx * K1X + K1X;        hy = by * K1Y + (h - 2 * K1X - K1Y); hr = h - 2 * K1X - K1Y + 1; hc = 2 + K1X; }
      halo_role = h < kHaloX2;
      halo_in = halo_role && hx >= 0 && hx < nxi && hy >= 0 && hy < nyi;
      hbr = hr; hbc = hc;                              // the ring and the boxes share their origin (x0-2, y0-1)
      pc0 = pc1 = pl0 = pl1 = a3l0 = a3l1 = 0.0;
    }
    const bool has_p = j < nz, has_mu = j >= 1;
    const int64_t ip = col + (int64_t)j * np;          // rows of plane j (p', x) ; plane j - 1 is ip - np (mu)
    // ---- 1. wait for the stage, read every operand of the step into registers
    mbar_wait(&sm.full[slot], (ph >> slot) & 1u);
    ph ^= 1u << slot;
    const ST& S = sm.st[slot];
    double2 ro = make_double2(0.0, 0.0), po = ro, dd = make_double2(1.0, 1.0), xo = xq0;
    double rh = 0.0, phh = 0.0, dh = 1.0;
    if (has_p) {
      ro = *reinterpret_cast<const double2*>(&S.vz[ty + 1][sc0]);
      po = *reinterpret_cast<const double2*>(&S.vp[ty + 1][sc0]);
      if (MIXED) dd = ldf2(reinterpret_cast<const float*>(&S.vd[ty + 1][ST::VDX + 2 * tx]));
      else dd = *reinterpret_cast<const double2*>(&S.vd[ty + 1][sc0]);
      if (halo_role) { rh = S.vz[hbr][hbc]; phh = S.vp[hbr][hbc]; dh = (double)S.vd[hbr][hbc + ST::VDX - 2]; }
      xq0 = xq1;                                                    // x for the p'-plane two steps ahead
      if (!do_x) {}
      else if (j + 2 < nz) { if (own) xq1 = ldd2(xg + ip + 2 * np); }
      else if (k + 1 < my_tiles) { bool on; const int64_t cn = tile_col(k + 1, &on); if (on) xq1 = ldd2(xg + cn + (int64_t)(j + 2 - nz) * np); }
    }
    double2 a1 = make_double2(0.0, 0.0), a2u = a1, a2l = a1, a3u = a1;
    double a1l = 0.0;
    if (has_mu) {
      a1 = k1_ld_pair<MIXED>(&S.m1[ty][AL1 + 2 * tx]);
      a1l = (double)S.m1[ty][AL1 + 2 * tx - 1];
      a2u = k1_ld_pair<MIXED>(&S.m2[ty + 1][2 * tx]);
      a2l = k1_ld_pair<MIXED>(&S.m2[ty][2 * tx]);
      a3u = k1_ld_pair<MIXED>(&S.m3[ty][2 * tx]);
    }
#if CUTH_K1_SPLIT
    // ---- 2. every warp has finished step s - 2 and has written its part of the ring plane of step s - 1
    if (s > 0) {
      mbar_wait(&sm.ringbar, (uint32_t)((s - 1) & 1));
      if (tid == 0 && s + kK1Stages - 1 < total) request_next();     // the stage of step s - 1 is consumed: refill it
    }
#else
    // ---- 2. plane j - 1 of the p' ring is complete, plane j - 2 no longer read, the stage is consumed
    __syncthreads();
    if (tid == 0 && s + kK1Stages < total) request_next();
#endif
    // ---- 3. plane j of p'
    double ph0 = 0.0, ph1 = 0.0;
    if (has_p) {
      if (own) {
        // fp32-stored operator: vd = 1/D0; fp64 operator: vd = D0, inverted in registers (rcp_diag: within an ulp)
        const double z0 = jac ? (MIXED ? ro.x * dd.x : ro.x * rcp_diag(dd.x)) : ro.x;
        const double z1 = jac ? (MIXED ? ro.y * dd.y : ro.y * rcp_diag(dd.y)) : ro.y;
        ph0 = fma(beta, po.x, z0); ph1 = fma(beta, po.y, z1);
        std2(p_out + ip, ph0, ph1);
        if (do_x) std2(xg + ip, fma(xalpha, po.x, xo.x), fma(xalpha, po.y, xo.y));
      }
      std2(&sm.sp[rw][ty + 1][sc0], ph0, ph1);
      if (halo_role) {
        const double zh = jac ? (MIXED ? rh * dh : rh * rcp_diag(dh)) : rh;
        sm.sp[rw][hr][hc] = halo_in ? fma(beta, phh, zh) : 0.0;
      }
    }
#if CUTH_K1_SPLIT
    __syncwarp();
    if (tx == 0) mbar_arrive(&sm.ringbar);             // phase s: this warp's part of the plane is written, its operands are read
#endif
    // ---- 4. rows of plane j - 1 of mu = A p'
    if (has_mu && own) {
      const double (*P)[XS] = sm.sp[rr];
      const double vl = P[ty + 1][sc0 - 1], vr = P[ty + 1][sc0 + 2];
      const double2 dn = *reinterpret_cast<const double2*>(&P[ty][sc0]);
      const double2 up = *reinterpret_cast<const double2*>(&P[ty + 2][sc0]);
      double m0, m1;
      if (!MIXED) {
        m0 = dcur.x * pc0;              m1 = dcur.y * pc1;
        m0 = fma(a1.x, pc1, m0);        m1 = fma(a1.x, pc0, m1);
        m0 = fma(a1l, vl, m0);          m1 = fma(a1.y, vr, m1);
        m0 = fma(a2u.x, up.x, m0);      m1 = fma(a2u.y, up.y, m1);
        m0 = fma(a2l.x, dn.x, m0);      m1 = fma(a2l.y, dn.y, m1);
        m0 = fma(a3u.x, ph0, m0);       m1 = fma(a3u.y, ph1, m1);
        m0 = fma(a3l0, pl0, m0);        m1 = fma(a3l1, pl1, m1);
      } else {
        const double sl = s_layer[j - 1];
        m0 = sl * pc0;                          m1 = sl * pc1;
        m0 = fma(a1.x, pc1 - pc0, m0);          m1 = fma(a1.x, pc0 - pc1, m1);
        m0 = fma(a1l, vl - pc0, m0);            m1 = fma(a1.y, vr - pc1, m1);
        m0 = fma(a2u.x, up.x - pc0, m0);        m1 = fma(a2u.y, up.y - pc1, m1);
        m0 = fma(a2l.x, dn.x - pc0, m0);        m1 = fma(a2l.y, dn.y - pc1, m1);
        m0 = fma(a3u.x, ph0 - pc0, m0);         m1 = fma(a3u.y, ph1 - pc1, m1);
        m0 = fma(a3l0, pl0 - pc0, m0);          m1 = fma(a3l1, pl1 - pc1, m1);
      }
      std2(mug + ip - np, m0, m1);
      dot = fma(pc0, m0, dot);
      dot = fma(pc1, m1, dot);
    }
    // ---- rotate
    pl0 = pc0; pl1 = pc1; pc0 = ph0; pc1 = ph1; a3l0 = a3u.x; a3l1 = a3u.y;
    if (!MIXED) dcur = dd;                             // D0 of plane j serves the mu rows of the next step
    if (++slot == kK1Stages) slot = 0;
    rr = rw;
    if (++rw == kK1Ring) rw = 0;
    if (++j == spt) { j = 0; ++k; }
  }
}

// K1 with TMA-staged operands.  tmP / tmP2: maps of the two direction buffers (ctl->pcur says which one is current).
__global__ void __launch_bounds__(kThreads, 2) k_fused_pspmv_tma(
    const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials, const __grid_constant__ CUtensorMap tmZ,
    const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmP2,
    const __grid_constant__ CUtensorMap tmDinv, const __grid_constant__ CUtensorMap tmD0,
    const __grid_constant__ CUtensorMap tmF1, const __grid_constant__ CUtensorMap tmF2,
    const __grid_constant__ CUtensorMap tmF3, const __grid_constant__ CUtensorMap tmE1,
    const __grid_constant__ CUtensorMap tmE2, const __grid_constant__ CUtensorMap tmE3) {
  extern __shared__ __align__(128) unsigned char k1_smem_raw[];
  if (ctl->halt) return;                     // unrolled graph body: this pass is over
  const Ctx c = *ctxp;
  if (c.k1_split && ctl->stage != 0) return; // thin stacks: the late stage belongs to k_fused_pspmv_x2 (cuth_api.cu make_plan)
  const int pcur = ctl->pcur;
  double* p_out = pcur ? c.p : c.p2;
  const CUtensorMap* tp = pcur ? &tmP2 : &tmP;
  const double beta = ctl->beta, xalpha = ctl->xalpha;
  double acc[1] = {0.0};
  double* red; int* flag;
  if (ctl->stage == 0) {
    K1Smem<true>& sm = *reinterpret_cast<K1Smem<true>*>(k1_smem_raw);
    fused_pspmv_tma_body<true>(c, sm, p_out, beta, xalpha, &tmZ, tp, &tmDinv, &tmF1, &tmF2, &tmF3, acc[0]);
    red = sm.red; flag = &sm.s_flag;
  } else {
    K1Smem<false>& sm = *reinterpret_cast<K1Smem<false>*>(k1_smem_raw);
    fused_pspmv_tma_body<false>(c, sm, p_out, beta, xalpha, &tmZ, tp, &tmD0, &tmE1, &tmE2, &tmE3, acc[0]);
    red = sm.red; flag = &sm.s_flag;
  }
  if (grid_sum_last_block<1>(acc, partials, &ctl->ticket[1], red, flag) && threadIdx.x == 0) {
    ctl->pcur = pcur ^ 1;
    policy_after_spmv(ctl, acc[0], true, &c);   // Alg. 1 line 7; x += alpha p deferred to the next K1 (or to K2: xnow)
  }
}

}  // namespace cuth
