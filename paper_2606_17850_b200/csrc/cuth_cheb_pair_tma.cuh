// cuth_cheb_pair_tma.cuh -- k_cheb_pair_f32 (two Chebyshev passes per kernel, see cuth_cheb_pair.cuh) with its
// global operands brought in by TMA.
//
// ncu on the LDG version: 54 % of the stall samples on the long scoreboard at 4 CTAs/SM, 0.59 of the HBM peak;
// prefetching into registers costs the occupancy it needs (123 registers, slower).  Here the operands of a plane
// -- U (region + the rows above and below), V, r and the three off-diagonals -- are boxes of 3-D tensors
// (x, y, z) that one thread requests with cp.async.bulk.tensor three planes ahead into a ring of shared-memory
// stages; completion is an mbarrier transaction count, no register holds a byte in flight.  Cells outside the
// grid are zero-filled by the TMA unit and the per-diagonal copies of the matrix have zero tails, so a missing
// neighbour is a zero value with a zero coefficient and the arithmetic needs no bounds predicate at all; only
// the two global stores are predicated.
//
// A stage is consumed in the W phase of step k (before the plane's one __syncthreads), so the same barrier
// that orders the W ring also frees the stage for the plane three steps ahead: no "empty" mbarriers.
// Requirements: nx a multiple of 16 bytes of elements (tensor-map strides), i.e. nx % 4 == 0 (fp32 A2) or
// nx % 8 == 0 (fp16 A3); otherwise cuth_api.cu keeps the LDG version.
#pragma once
#include <cuda.h>
#include "cuth_cheb_pair.cuh"

namespace cuth {

constexpr int kPairStages = 3;

// The innermost coordinate of a TMA box must be a multiple of 16 bytes (measured: an 8-byte offset is an
// illegal-instruction fault), the region origin x0 = 60 bx - 2 is not: a box starts at x0 rounded down to 16 bytes
// and is 16 bytes wider than the region; the thread's pair then sits at column (x0 - start) + 2 tx of the row.
template <class E> struct PairBox {
  static constexpr int AL = 16 / (int)sizeof(E);     // elements per 16 bytes
  static constexpr int W = QX + AL;                  // box width in elements
};
// RY = rows of the region (one warp each): 8 (256 threads, 4 CTAs/SM, 360 of 512 cells interior) or 16 (512
// threads, 2 CTAs/SM, 840 of 1024 interior: a sixth less recomputation for the same number of resident warps).
template <class E, int RY>
struct PairStage {                         // every member starts on a 128-byte boundary (TMA destination)
  alignas(128) float u[RY + 2][PairBox<float>::W];   // rows y0-1 .. y0+RY of U
  alignas(128) float v[RY][PairBox<float>::W];
  alignas(128) float r[RY][PairBox<float>::W];
  alignas(128) E f1[RY][PairBox<E>::W];
  alignas(128) E f2[RY + 1][PairBox<E>::W];          // rows y0-1 .. y0+RY-1: the entry towards y-1 is the row above's
  alignas(128) E f3[RY][PairBox<E>::W];
  // bytes the six boxes deliver (the padding between members is not part of any box)
  static constexpr uint32_t kTxBytes = sizeof(float) * PairBox<float>::W * (RY + 2 + RY + RY) +
                                       sizeof(E) * PairBox<E>::W * (RY + RY + 1 + RY);
};
// dynamic shared memory of the kernel: stages | W ring | mbarriers | reduction scratch | flag
template <class E, int RY>
struct PairSmem {
  PairStage<E, RY> st[kPairStages];
  alignas(8) float sW[2][RY][QX];
  alignas(8) uint64_t full[kPairStages];
  double red[32];
  int s_flag;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, uint64_t* bar, int x, int y, int z) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(tm)), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
      : "memory");
}

// a pair of x-neighbours of a shared-memory row, promoted to fp32 (and rescaled for the fp16 copy)
__device__ __forceinline__ float2 lds_pair(const float* p, float) { return *reinterpret_cast<const float2*>(p); }
__device__ __forceinline__ float2 lds_pair(const __half* p, float s) {
  const float2 f = __half22float2(*reinterpret_cast<const __half2*>(p));
  return make_float2(f.x * s, f.y * s);
}

// LAST = true: the second pass is the last one of the apply (k_cheb_last's job): Y = Z_k goes to the fp64 vector
// z of the outer loop, rho = r.z is reduced over the grid and the epilogue forms beta; W = Z_{k-1} is not stored.
template <class M, bool LAST, int RY>
__global__ void __launch_bounds__(32 * RY, RY == 8 ? 4 : 2) k_cheb_pair_tma(
    const Ctx* __restrict__ ctxp, Ctl* ctl, double* partials, int step, int wout, int yout,
    const __grid_constant__ CUtensorMap tmU,
    const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmR,
    const __grid_constant__ CUtensorMap tm1, const __grid_constant__ CUtensorMap tm2,
    const __grid_constant__ CUtensorMap tm3) {
  using E = typename M::elem;
  extern __shared__ __align__(128) unsigned char pair_smem_raw[];
  PairSmem<E, RY>& sm = *reinterpret_cast<PairSmem<E, RY>*>(pair_smem_raw);
  PairStage<E, RY>* st = sm.st;
  float (*sW)[RY][QX] = sm.sW;
  uint64_t* full = sm.full;
  constexpr int QIYr = RY - 2;                        // interior rows written by this CTA
  const DiaDev& A = ctxp->A;
  const float c1a = (float)ctxp->cheb_c1[step], c2a = (float)ctxp->cheb_c2[step];
  const float c1b = (float)ctxp->cheb_c1[step + 1], c2b = (float)ctxp->cheb_c2[step + 1];
  float* __restrict__ Wg = (float*)ctxp->cd[LAST ? 0 : wout];
  float* __restrict__ Yg = (float*)ctxp->cd[LAST ? 0 : yout];
  double* __restrict__ Zg = ctxp->cz;                 // LAST: z = Z_k in fp64
  const double* __restrict__ R64 = ctxp->r;           // LAST: r in fp64 for rho = r.z
  __builtin_assume(__isGlobal(Wg)); __builtin_assume(__isGlobal(Yg));
  __builtin_assume(__isGlobal(Zg)); __builtin_assume(__isGlobal(R64));
  double acc = 0.0;
  const double* __restrict__ s_layer = A.s_layer;
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  const int nxi = (int)A.nx, nyi = A.ny, nz = A.nz;
  const int tiles_x = (nxi + QIX - 1) / QIX, tiles_y = (nyi + QIYr - 1) / QIYr;
  const int ntiles = tiles_x * tiles_y;
  const int64_t nx = A.nx, np = A.nxny;
  const float ms = M::inv(A);
  const float2 z2 = make_float2(0.f, 0.f);
  const bool rim = tx == 0 || tx == 31 || ty == 0 || ty == RY - 1;
  constexpr unsigned kAll = 0xffffffffu;
  constexpr uint32_t kStageBytes = PairStage<E, RY>::kTxBytes;

  if (tid == 0) {
    for (int s = 0; s < kPairStages; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  uint32_t ph = 0;                         // bit S: parity of the next fill of stage S to wait for
  for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const int bx = t % tiles_x, by = t / tiles_x;
    const int x0 = bx * QIX - 2, y0 = by * QIYr - 1;                   // region origin (x0 even)
    const int x = x0 + 2 * tx, y = y0 + ty;
    const bool inner = !rim && x >= 0 && x < nxi && y >= 0 && y < nyi;  // nx even: x + 1 < nx with x
    const int64_t c0 = inner ? x + nx * (int64_t)y : 0;
    float* pW = Wg + c0; float* pY = Yg + c0 - np;                       // Y trails W by a plane
    double* pZ = Zg + c0 - np; const double* pR = R64 + c0 - np;

    // box starts: x0 rounded down to 16 bytes of elements (two's complement & works for x0 = -2 too)
    const int xs_f = x0 & ~(PairBox<float>::AL - 1), xs_e = x0 & ~(PairBox<E>::AL - 1);
    const int cf = (x0 - xs_f) + 2 * tx, ce = (x0 - xs_e) + 2 * tx;    // this thread's pair inside a staged row
    // Plane kp lives in stage kp % 3 (every tile starts at stage 0, so the stage of a step is a compile-time
    // constant in the three-fold unrolled march below); ph holds, per stage, the parity of its next fill.
    auto request = [&](auto stage_t, int kp) {   // thread 0: the six boxes of plane kp into stage S
      constexpr int S = decltype(stage_t)::value;
      mbar_expect_tx(&full[S], kStageBytes);
      tma_load_3d(st[S].u, &tmU, &full[S], xs_f, y0 - 1, kp);
      tma_load_3d(st[S].v, &tmV, &full[S], xs_f, y0, kp);
      tma_load_3d(st[S].r, &tmR, &full[S], xs_f, y0, kp);
      tma_load_3d(st[S].f1, &tm1, &full[S], xs_e, y0, kp);
      tma_load_3d(st[S].f2, &tm2, &full[S], xs_e, y0 - 1, kp);
      tma_load_3d(st[S].f3, &tm3, &full[S], xs_e, y0, kp);
    };
    auto arrived = [&](auto stage_t) {     // everybody: block until the pending fill of stage S has landed
      constexpr int S = decltype(stage_t)::value;
      mbar_wait(&full[S], (ph >> S) & 1u);
      ph ^= 1u << S;
    };
    constexpr std::integral_constant<int, 0> S0{};
    constexpr std::integral_constant<int, 1> S1{};
    constexpr std::integral_constant<int, 2> S2{};

    __syncthreads();                       // the previous tile's stages and W ring are dead
    if (tid == 0) {
      request(S0, 0);
      request(S1, 1);                      // nz >= 2
      if (nz > 2) request(S2, 2);
    }

    arrived(S0);
    float2 u_lo = z2, u_c = lds_pair(&st[0].u[ty + 1][cf], 1.f);        // U on planes k-1, k
    float2 w_lo = z2, w_c = z2;                                         // W on planes k-2, k-1
    float2 a3l_w = z2, a3l_y = z2;                                      // D3 below plane k / below plane k-1
    float pf1l = 0.f, pf1a = 0.f, pf1b = 0.f, ps = 0.f;                 // row of plane k-1, kept for Y
    float2 pf2u = z2, pf2l = z2, pa3u = z2, pr = z2;

    // One step of the march: W on plane k from stage S (HAS_W), the barrier, Y on plane k-1.
    auto do_step = [&](auto stage_t, auto has_w_t, int k) {
      constexpr int S = decltype(stage_t)::value, SN = (S + 1) % kPairStages;
      constexpr bool HAS_W = decltype(has_w_t)::value;
      float2 w = z2, u_hi = z2, rv = z2, f1p = z2, f2u = z2, f2l = z2, a3u = z2;
      float f1l = 0.f, s = 0.f;
      double2 rd = make_double2(0.0, 0.0);
      if (LAST && inner && k >= 1) rd = *reinterpret_cast<const double2*>(pR);   // for Y below; flies during W
      if (HAS_W) {
        // ---- W on plane k: operands from the stage (no bounds predicates: absent = zero x zero)
        const PairStage<E, RY>& T = st[S];
        const float2 v2u = lds_pair(&T.u[ty + 2][cf], 1.f), v2l = lds_pair(&T.u[ty][cf], 1.f);
        const float2 zo = lds_pair(&T.v[ty][cf], 1.f);
        rv = lds_pair(&T.r[ty][cf], 1.f);
        f1p = lds_pair(&T.f1[ty][ce], ms);
        f2u = lds_pair(&T.f2[ty + 1][ce], ms); f2l = lds_pair(&T.f2[ty][ce], ms);
        a3u = lds_pair(&T.f3[ty][ce], ms);
        if (k + 1 < nz) {
          arrived(std::integral_constant<int, SN>{});
          u_hi = lds_pair(&st[SN].u[ty + 1][cf], 1.f);
        }
        const float vl = __shfl_up_sync(kAll, u_c.y, 1), vr = __shfl_down_sync(kAll, u_c.x, 1);
        f1l = __shfl_up_sync(kAll, f1p.y, 1);
        s = (float)s_layer[k];
        float a0 = s * u_c.x, a1 = s * u_c.y;
        a0 += f1p.x * (u_c.y - u_c.x);   a1 += f1p.x * (u_c.x - u_c.y);
        a0 += f1l * (vl - u_c.x);        a1 += f1p.y * (vr - u_c.y);
        a0 += f2u.x * (v2u.x - u_c.x);   a1 += f2u.y * (v2u.y - u_c.y);
        a0 += f2l.x * (v2l.x - u_c.x);   a1 += f2l.y * (v2l.y - u_c.y);
        a0 += a3u.x * (u_hi.x - u_c.x);  a1 += a3u.y * (u_hi.y - u_c.y);
        a0 += a3l_w.x * (u_lo.x - u_c.x); a1 += a3l_w.y * (u_lo.y - u_c.y);
        w = make_float2(u_c.x + c1a * (u_c.x - zo.x) + c2a * (rv.x - a0),
                        u_c.y + c1a * (u_c.y - zo.y) + c2a * (rv.y - a1));
        if (!LAST && inner) *reinterpret_cast<float2*>(pW) = w;
      }
      __syncthreads();                     // W(k-1) complete, W(k-2) no longer read, stage of plane k consumed
      if (HAS_W) {
        if (tid == 0 && k + kPairStages < nz) request(stage_t, k + kPairStages);
        *reinterpret_cast<float2*>(&sW[k & 1][ty][2 * tx]) = w;
      }
      if (k >= 1) {
        // ---- Y on plane k-1
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
          const float y0v = w_c.x + c1b * (w_c.x - u_lo.x) + c2b * (pr.x - a0);
          const float y1v = w_c.y + c1b * (w_c.y - u_lo.y) + c2b * (pr.y - a1);
          if (LAST) {
            const double zk0 = (double)y0v, zk1 = (double)y1v;
            *reinterpret_cast<double2*>(pZ) = make_double2(zk0, zk1);
            acc = fma(rd.x, zk0, acc);
            acc = fma(rd.y, zk1, acc);
          } else {
            *reinterpret_cast<float2*>(pY) = make_float2(y0v, y1v);
          }
        }
      }
      // ---- rotate: plane k becomes plane k-1
      a3l_y = pa3u;
      pf1l = f1l; pf1a = f1p.x; pf1b = f1p.y; ps = s; pf2u = f2u; pf2l = f2l; pa3u = a3u; pr = rv;
      w_lo = w_c; w_c = w;
      a3l_w = a3u;
      u_lo = u_c; u_c = u_hi;
      pW += np; pY += np; pZ += np; pR += np;
    };
    constexpr std::true_type HW{};
    constexpr std::false_type NW{};
    int k = 0;
    for (; k + kPairStages <= nz; k += kPairStages) {
      do_step(S0, HW, k); do_step(S1, HW, k + 1); do_step(S2, HW, k + 2);
    }
    // the last nz % 3 planes, then the step that only forms Y on the top plane
    if (k < nz) {
      do_step(S0, HW, k); ++k;
      if (k < nz) { do_step(S1, HW, k); ++k; do_step(S2, NW, k); }
      else do_step(S1, NW, k);
    } else {
      do_step(S0, NW, k);
    }
  }
  if (LAST) {
    double a[1] = {acc};
    if (grid_sum_last_block<1>(a, partials + 3 * kMaxBlocks, &ctl->ticket[5], sm.red, &sm.s_flag) && tid == 0) {
      const double rho_new = a[0];
      ctl->beta = ctl->beta_zero ? 0.0 : rho_new / ctl->rho;     // Alg. 1 line 11 (line 3 when restarting)
      ctl->rho = rho_new;
      ctl->beta_zero = 0;
      if (!(rho_new == rho_new) || rho_new <= 0.0) ctl->status = CUTH_SOLVE_BREAKDOWN;   // q(A) not SPD: bad interval
    }
  }
}

}  // namespace cuth
