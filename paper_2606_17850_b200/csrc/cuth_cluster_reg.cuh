// cuth_cluster_reg.cuh -- the cluster-resident PCG solve of cuth_cluster.cuh with the ROW STATE IN REGISTERS, for grids of
// at most 1024 rows per CTA (BASELINE cfg 1: 8 192 rows = 8 CTAs x 1024).
//
// Why: of the 8 600 cycles of an iteration of k_pcg_cluster at cfg 1, 2 300 are the fused direction +
// SpMV phase -- 27 shared-memory loads per row, of which only the neighbours' z and p have to come from shared memory --
// and 1 350 are the scalar policy code walking a control block in shared memory.  Here
//   * a thread owns two rows (512 threads, a 128-register budget) and keeps their seven coefficients, the six neighbour
//     ADDRESSES (32-bit shared::cluster addresses from mapa, formed once), r, x, 1/D0 and mu in registers;
//   * z and p of a row sit side by side as one 16-byte pair {z, p}: a neighbour costs ONE ld.shared::cluster.v2.f64, a row
//     seven 16-byte loads instead of 27 8-byte ones; there are two pair buffers: the iteration reads PB[cur] and writes
//     {z', p'} of its own rows into PB[cur ^ 1] with one 16-byte store, so the two barriers per iteration of
//     cuth_cluster.cuh remain two;
//   * the scalars of the common case (alpha, beta, rho, the iteration counters, the stopping / evaluation tests) live in
//     registers of every thread -- identical everywhere, because every thread adds the same partial sums in the same
//     order; the control block in shared memory is touched only when something happens (an evaluation of the true
//     residual is due, convergence, breakdown, the cap): then the registers are written back and the SAME policy
//     functions as everywhere else (cuth_policy.cuh) run, exactly as in cuth_cluster.cuh;
//   * the true-residual phase exchanges x through the pair buffer that is dead at that point.
// Same arithmetic per row, in the same order, as cuth_cluster.cuh (hence as the flat kernels); only the order in which the
// rows are summed differs.  FP64 and MIXED (difference form), M = diag A or I, steady and transient, batched.
#pragma once
#include "cuth_cluster.cuh"

namespace cuth {

constexpr int kCrRows = 2;                               // rows per thread
constexpr int kCrMaxThreads = 512;                       // 512 threads x 2 rows = 1024 rows per CTA at most
constexpr int kCrBytesPerRow = 32;                       // two {z, p} pairs

inline size_t cluster_reg_smem_bytes(int64_t rows_per_cta) {
  return (size_t)kClusterFixedBytes + (size_t)kCrBytesPerRow * (size_t)rows_per_cta;
}
inline bool cluster_reg_fits(int64_t nx, int64_t ny, int64_t nz, int nc, int threads = kCrMaxThreads) {
  return cluster_rows_per_cta(nx, ny, nz, nc) <= threads * kCrRows;
}

#ifdef __CUDACC__

__device__ __forceinline__ double2 cl_ld_pair(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

__device__ __forceinline__ double2 ld_own_pair(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}

template <int NC, int NT>
__global__ void __launch_bounds__(NT, 1) k_pcg_cluster_reg(const Ctx* __restrict__ ctxp, Ctl* ctl_g, int rows_per_cta) {
  constexpr int NW = NT / 32;
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) unsigned char cl_raw[];
  ClusterSmem* sm = reinterpret_cast<ClusterSmem*>(cl_raw);
  const int R = rows_per_cta;
  ctxp += blockIdx.x / NC;                             // batched use: one cluster per right-hand side
  ctl_g += blockIdx.x / NC;
  double2* PB = reinterpret_cast<double2*>(cl_raw + kClusterFixedBytes);     // [2][R] pairs {z, p}
  const uint32_t pb_stride = (uint32_t)R * 16u;                              // bytes between the two pair buffers
  {
    const uint64_t* src = reinterpret_cast<const uint64_t*>(ctxp);
    uint64_t* dst = reinterpret_cast<uint64_t*>(&sm->ctx);
    for (int q = threadIdx.x; q < (int)(sizeof(Ctx) / 8); q += NT) dst[q] = src[q];
    __syncthreads();
  }
  const Ctx& c = sm->ctx;
  const DiaDev& A = c.A;
  const int64_t n = A.n, nx = A.nx, np = A.nxny;
  const int nxi = (int)A.nx, nyi = A.ny, nzi = A.nz;
  const unsigned me = cluster.block_rank();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  Ctl* my = &sm->ctl[wid];
  const bool jac = c.jacobi != 0;
  int parity = 0;
  // ---- ownership: slabs along y or z, as cuth_cluster.cuh
  const ClusterSplit sp = cluster_split(nyi, nzi);
  auto slab0 = [&](int q) { return (int)(((int64_t)q * sp.len) / NC); };
  auto owner_of = [&](int u) {
    int q = (int)(((int64_t)u * NC) / sp.len);
    while (q + 1 < NC && slab0(q + 1) <= u) ++q;
    while (q > 0 && slab0(q) > u) --q;
    return q;
  };
  const int s0 = slab0((int)me), s1 = slab0((int)me + 1);
  const int hy = sp.axis_z ? nyi : s1 - s0, hz = sp.axis_z ? s1 - s0 : nzi;
  const int my_rows = nxi * hy * hz;                   // <= R <= 1024
  auto local_of = [&](int q, int x, int y, int z) {
    const int a0 = slab0(q), a1 = slab0(q + 1);
    return sp.axis_z ? x + nxi * (y + nyi * (z - a0)) : x + nxi * ((y - a0) + (a1 - a0) * z);
  };

  // ---- the thread's rows: l = threadIdx.x + q * 512
  bool has[kCrRows];
  int gi[kCrRows];                                     // global row
  uint32_t own[kCrRows];                               // shared::cta address of the row's pair in PB[0]
  uint32_t nb[kCrRows][6];                             // shared::cluster addresses of the six neighbours' pairs in PB[0]
  double cf[kCrRows][7];                               // c0 (D0, or s(z) in the early stage), six off-diagonal coefficients
  double rr_[kCrRows], xx[kCrRows], di[kCrRows], mu[kCrRows], pn[kCrRows], zr[kCrRows];   // zr, pn: the row's own {z, p}
  // where p' of the x+1 / x-1 neighbour comes from: 0 = absent (own value, coefficient 0), 1 = the adjacent lane
  // (it holds the neighbouring row: same fma on the same operands, shuffled instead of recomputed), 2 = another warp's
  // row: recomputed from its pair
  int xpm[kCrRows], xmm[kCrRows];
  const uint32_t pb0 = cl_smem_u32(PB);
#pragma unroll
  for (int q = 0; q < kCrRows; ++q) {
    const int l = (int)threadIdx.x + q * NT;
    has[q] = l < my_rows;
    const int ll = has[q] ? l : 0;
    const int x = ll % nxi, t = ll / nxi, u = t % hy, v = t / hy;
    const int y = sp.axis_z ? u : u + s0, z = sp.axis_z ? v + s0 : v;
    gi[q] = (int)(x + nx * (y + (int64_t)nyi * z));
    own[q] = pb0 + 16u * (uint32_t)ll;
    // neighbours in the order of Alg. 2 as the flat kernels add them: +1, -1, +nx, -nx, +nx*ny, -nx*ny; an absent one
    // is replaced by the row itself (its coefficient is a stored structural zero)
    const int dx[6] = {1, -1, 0, 0, 0, 0}, dy[6] = {0, 0, 1, -1, 0, 0}, dz[6] = {0, 0, 0, 0, 1, -1};
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const int xn = x + dx[k], yn = y + dy[k], zn = z + dz[k];
      unsigned q_own = me; int idx = ll;
      if (xn >= 0 && xn < nxi && yn >= 0 && yn < nyi && zn >= 0 && zn < nzi) {
        q_own = (unsigned)owner_of(sp.axis_z ? zn : yn);
        idx = local_of((int)q_own, xn, yn, zn);
      }
      nb[q][k] = cl_mapa(pb0 + 16u * (uint32_t)idx, q_own);
    }
    xpm[q] = (!has[q] || x + 1 >= nxi) ? 0 : ((threadIdx.x & 31) < 31 ? 1 : 2);
    xmm[q] = (!has[q] || x == 0) ? 0 : ((threadIdx.x & 31) > 0 ? 1 : 2);
    di[q] = (has[q] && jac) ? A.dinv[gi[q]] : 1.0;
    xx[q] = has[q] ? c.x[gi[q]] : 0.0;
    rr_[q] = 0.0; mu[q] = 0.0; pn[q] = 0.0; zr[q] = 0.0;
  }
  auto load_coefs = [&](bool early) {
#pragma unroll
    for (int q = 0; q < kCrRows; ++q) {
      const int64_t i = gi[q];
      const bool h = has[q];
      const bool up1 = h && i + 1 < n, lo1 = h && i >= 1, up2 = h && i + nx < n, lo2 = h && i >= nx, up3 = h && i + np < n,
                 lo3 = h && i >= np;
      if (early) {          // fp32-stored off-diagonals promoted to fp64, difference form: c0 = s(z)
        cf[q][0] = h ? A.s_layer[(unsigned)i / (unsigned)np] : 0.0;
        cf[q][1] = up1 ? (double)A.f1[i] : 0.0; cf[q][2] = lo1 ? (double)A.f1[i - 1] : 0.0;
        cf[q][3] = up2 ? (double)A.f2[i] : 0.0; cf[q][4] = lo2 ? (double)A.f2[i - nx] : 0.0;
        cf[q][5] = up3 ? (double)A.f3[i] : 0.0; cf[q][6] = lo3 ? (double)A.f3[i - np] : 0.0;
      } else {
        cf[q][0] = h ? A.d0[i] : 0.0;
        cf[q][1] = up1 ? A.d1[i] : 0.0; cf[q][2] = lo1 ? A.d1[i - 1] : 0.0;
        cf[q][3] = up2 ? A.d2[i] : 0.0; cf[q][4] = lo2 ? A.d2[i - nx] : 0.0;
        cf[q][5] = up3 ? A.d3[i] : 0.0; cf[q][6] = lo3 ? A.d3[i - np] : 0.0;
      }
    }
  };
  // (A1 x)_row with x exchanged through pair buffer `buf` (its .x members); the fp64 coefficients must be loaded
  auto apply_x = [&](int q, uint32_t boff) {
    double vk[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) vk[k] = cl_ld_pair(nb[q][k] + boff).x;
    double acc = cf[q][0] * xx[q];
#pragma unroll
    for (int k = 0; k < 6; ++k) acc = fma(cf[q][k + 1], vk[k], acc);
    return acc;
  };
  auto st_pair = [&](int q, uint32_t boff, double a, double b) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(own[q] + boff), "d"(a), "d"(b) : "memory");
  };
  if (lane == 0) *my = *ctl_g;                         // cleared by k_set_ctx
  if (threadIdx.x == 0) {
    cluster_bars_init(sm);
  }
  load_coefs(false);                                   // r0 = b - A1 x0 needs the fp64 operator
#pragma unroll
  for (int q = 0; q < kCrRows; ++q) if (has[q]) { st_pair(q, pb_stride, xx[q], 0.0); st_pair(q, 0u, 0.0, 0.0); }
  cluster.sync();

  // ---- Alg. 1 lines 1-3: r0 = b - A1 x0, z0 = M^-1 r0 -> PB[0] = {z0, 0}; beta = 0 makes the first p' = z0
  {
    double acc[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int q = 0; q < kCrRows; ++q) if (has[q]) {
      const double bi = c.b[gi[q]];
      const double ri = bi - apply_x(q, pb_stride);
      const double zi = jac ? ri * di[q] : ri;
      rr_[q] = ri; zr[q] = zi;
      st_pair(q, 0u, zi, 0.0);
      acc[0] = fma(ri, zi, acc[0]); acc[1] = fma(ri, ri, acc[1]); acc[2] = fma(bi, bi, acc[2]);
    }
    cluster_allreduce<NC, 3, NW>(cluster, sm, acc, parity);
    if (lane == 0) my->want_true = (int)policy_init(my, c, acc[0], acc[1], acc[2]);      // want_true reused as "go"
    __syncwarp();
  }
  bool go = my->want_true != 0;
  bool early = my->stage == 0;
  if (go && early) load_coefs(true);
  uint32_t cur = 0u;                                   // byte offset of the CURRENT pair buffer: 0 or pb_stride
  // ---- the scalars of the common case, identical in every thread (see the header); written back to the control block
  //      before any policy function runs
  double rho = my->rho, beta = my->beta, alpha = 0.0, pAp = 0.0;
  int it = my->it, since = my->since_eval;
  const double tol2 = my->tol2, sw2 = my->sw2;
  const int period = c.period, max_iters = c.max_iters;
  bool broken = false;
#ifdef CUTH_CLUSTER_PROF
  long long ar[6] = {0, 0, 0, 0, 0, 0};
  long long tk[6] = {0, 0, 0, 0, 0, 0}, t0 = clock64(); unsigned long long g0; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g0)); int nit = 0;
#define CRK(i) { long long t1 = clock64(); tk[i] += t1 - t0; t0 = t1; }
#else
#define CRK(i)
#endif

  while (go) {
    // ---- AB: p' = z + beta p at the row and its six neighbours, mu = A p', p'.mu  (Alg. 1 lines 12 + 6)
    double a1[1] = {0.0};
    double pi[kCrRows];
#pragma unroll
    for (int q = 0; q < kCrRows; ++q) pi[q] = has[q] ? fma(beta, pn[q], zr[q]) : 0.0;      // the row's own {z, p} never left the registers
#pragma unroll
    for (int q = 0; q < kCrRows; ++q) {
      const double from_up = __shfl_down_sync(0xffffffffu, pi[q], 1), from_dn = __shfl_up_sync(0xffffffffu, pi[q], 1);
      if (has[q]) {
        double2 vk[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) vk[k] = cl_ld_pair(nb[q][k + 2] + cur);
        double pxp = xpm[q] == 1 ? from_up : pi[q], pxm = xmm[q] == 1 ? from_dn : pi[q];
        if (xpm[q] == 2) { const double2 v = cl_ld_pair(nb[q][0] + cur); pxp = fma(beta, v.y, v.x); }
        if (xmm[q] == 2) { const double2 v = cl_ld_pair(nb[q][1] + cur); pxm = fma(beta, v.y, v.x); }
        double acc = cf[q][0] * pi[q];
        acc = fma(cf[q][1], early ? pxp - pi[q] : pxp, acc);
        acc = fma(cf[q][2], early ? pxm - pi[q] : pxm, acc);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const double pk = fma(beta, vk[k].y, vk[k].x);
          acc = fma(cf[q][k + 3], early ? pk - pi[q] : pk, acc);
        }
        pn[q] = pi[q]; mu[q] = acc;
        a1[0] = fma(pi[q], acc, a1[0]);
      }
    }
    CRK(0)
    cluster_allreduce<NC, 1, NW>(cluster, sm, a1, parity);
    CRK(1)
    pAp = a1[0];
    if (!(pAp > 0.0) || !(pAp <= 1.79e308) || !(rho == rho)) {        // breakdown: the control block takes over
      if (lane == 0) { my->rho = rho; my->beta = beta; my->it = it; my->since_eval = since; policy_after_spmv(my, pAp, false); }
      __syncwarp();
      alpha = my->alpha; broken = true;
    } else {
      alpha = rho / pAp;                                              // Alg. 1 line 7 (policy_after_spmv)
    }
    CRK(2)
    // ---- C: x, r, z, dots; {z', p'} -> the other pair buffer
    double a2[2] = {0.0, 0.0};
#pragma unroll
    for (int q = 0; q < kCrRows; ++q) if (has[q]) {
      xx[q] = fma(alpha, pn[q], xx[q]);
      const double s0r = fma(-alpha, mu[q], rr_[q]);
      const double z0 = jac ? s0r * di[q] : s0r;
      rr_[q] = s0r; zr[q] = z0;
      st_pair(q, cur ^ pb_stride, z0, pn[q]);
      a2[0] = fma(s0r, z0, a2[0]); a2[1] = fma(s0r, s0r, a2[1]);
    }
    cur ^= pb_stride;
    CRK(3)
#ifdef CUTH_CLUSTER_PROF
    cluster_allreduce<NC, 2, NW>(cluster, sm, a2, parity, ar);
#else
    cluster_allreduce<NC, 2, NW>(cluster, sm, a2, parity);
#endif
    CRK(4)
    // ---- Alg. 1 lines 11, 13 and "is anything due?" -- policy_after_update's tests on registers
    {
      const double rho_new = a2[0], rr = a2[1];
      const int it1 = it + 1, since1 = since + 1;
      const bool due = broken || rr <= tol2 || (early && (rr <= sw2 || since1 >= period)) || it1 >= max_iters ||
                       !(rr == rr) || !(rho_new == rho_new);
      if (!due) {
        beta = rho_new / rho; rho = rho_new; it = it1; since = since1;
#ifdef CUTH_CLUSTER_PROF
        ++nit;
#endif
        CRK(5)
        continue;
      }
      if (lane == 0) {
        my->rho = rho; my->beta = beta; my->it = it; my->since_eval = since; my->pAp = pAp;
        if (!broken) my->alpha = alpha;
        unsigned g_, w_;
        policy_after_update(my, c, rho_new, rr, g_, w_);
        my->exiting = (int)g_;
      }
      __syncwarp();
      go = my->exiting != 0;
    }
    if (my->want_true) {
      // ---- D: true residual t = b - A1 x; x travels through the pair buffer that is dead now (the one AB read)
      const uint32_t dead = cur ^ pb_stride;
      if (early) load_coefs(false);
#pragma unroll
      for (int q = 0; q < kCrRows; ++q) if (has[q]) st_pair(q, dead, xx[q], 0.0);
      cluster.sync();
      double a3[2] = {0.0, 0.0};
      double tq[kCrRows];
#pragma unroll
      for (int q = 0; q < kCrRows; ++q) {
        tq[q] = 0.0;
        if (has[q]) {
          const double ti = c.b[gi[q]] - apply_x(q, dead);
          const double dd = ti - rr_[q];
          tq[q] = ti;
          a3[0] = fma(ti, ti, a3[0]); a3[1] = fma(dd, dd, a3[1]);
        }
      }
      cluster_allreduce<NC, 2, NW>(cluster, sm, a3, parity);
      if (lane == 0) my->exiting = (int)policy_after_true(my, c, a3[0], a3[1]);
      __syncwarp();
      go = my->exiting != 0;
      const int mode = my->restart;
      early = my->stage == 0;
      if (go && early) load_coefs(true);               // still early: back to the fp32-stored coefficients
      if (go && mode) {
        // ---- E: r := t, z = M^-1 r into the current pair buffer (p stays: nobody reads the buffer before the barrier)
        double a4[2] = {0.0, 0.0};
#pragma unroll
        for (int q = 0; q < kCrRows; ++q) if (has[q]) {
          const double ri = tq[q];
          const double zi = jac ? ri * di[q] : ri;
          rr_[q] = ri; zr[q] = zi;
          st_pair(q, cur, zi, pn[q]);
          a4[0] = fma(ri, zi, a4[0]); a4[1] = fma(ri, ri, a4[1]);
        }
        cluster_allreduce<NC, 2, NW>(cluster, sm, a4, parity);
        if (lane == 0) policy_after_restart(my, c, mode, a4[0], a4[1]);
        __syncwarp();
      }
    }
    // ---- back to the registers
    rho = my->rho; beta = my->beta; it = my->it; since = my->since_eval;
    broken = false;
#ifdef CUTH_CLUSTER_PROF
    ++nit;
#endif
    CRK(5)
  }
#ifdef CUTH_CLUSTER_PROF
  if ((threadIdx.x == 0 || threadIdx.x == 480) && blockIdx.x < NC) { unsigned long long g1; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g1));
    printf("cluster_reg prof cta %d thread %d NC=%d rows=%d its=%d ns/it=%.1f cyc/it: AB %.0f red1 %.0f pol1 %.0f C %.0f red2 %.0f pol2 %.0f | red2: tree %.0f bar %.0f tree2 %.0f send %.0f wait %.0f sum %.0f\n", (int)me, (int)threadIdx.x, NC, my_rows, nit, (double)(g1 - g0) / nit,
           (double)tk[0] / nit, (double)tk[1] / nit, (double)tk[2] / nit, (double)tk[3] / nit, (double)tk[4] / nit, (double)tk[5] / nit,
           (double)ar[0] / nit, (double)ar[1] / nit, (double)ar[2] / nit, (double)ar[3] / nit, (double)ar[4] / nit, (double)ar[5] / nit); }
#endif
  // ---- epilogue: x back to the caller's buffer, result record
  if (!my->refused) {
    const bool zero = my->zero_rhs != 0;
#pragma unroll
    for (int q = 0; q < kCrRows; ++q) if (has[q]) c.x[gi[q]] = zero ? 0.0 : xx[q];
  }
  if (me == 0 && threadIdx.x == 0) {
    my->exiting = 0;
    write_result(my, c);
    *ctl_g = *my;
  }
  cluster.sync();                                      // no CTA may exit while others still read its shared memory
}

#endif  // __CUDACC__

}  // namespace cuth
