// cuth_cluster.cuh -- the whole PCG solve inside ONE thread-block cluster, for grids small enough to live in the
// distributed shared memory of 8 or 16 SMs (BASELINE cfg 1: 8 192 unknowns).
//
// Why: on such grids the persistent kernel of cuth_persistent.cuh is pure barrier latency -- three grid-wide barriers
// of ~2 us per iteration through L2 (7.0 us per iteration at 8 k rows, HBM 2.5 % busy).  A cluster has
// a HARDWARE barrier (barrier.cluster) and its CTAs read and write each other's shared memory directly, so nothing
// of the iteration touches L2:
//   * CTA c owns a slab of the grid (along y or z): the r, z = M^-1 r, x, mu, 1/D0 and both copies of p of its rows,
//     the seven coefficients of each row and the (owner, index) of its six neighbours sit in its shared memory
//     (136 B per row);
//   * phase AB (Alg. 1 lines 12 + 6): a row forms p' = z + beta p for itself AND its six neighbours from their z and
//     old p -- read through distributed shared memory when a neighbour belongs to another CTA -- and applies A; the
//     same fma on the same operands as the neighbour's owner, hence the same bits; p' goes to the other p buffer, so
//     there is no barrier between the direction update and the SpMV: TWO cluster barriers per iteration;
//   * reductions: warp shuffle -> shared -> warp 0 -> every CTA's partial is STORED into all CTAs' shared memory
//     (remote stores) followed by a remote mbarrier arrive; every thread waits on its own CTA's mbarrier and adds the
//     partials in the same fixed order: all threads of all CTAs hold identical sums, no scalar is ever broadcast, and
//     the all-reduce doubles as the cluster-wide barrier of the phase (no barrier.cluster in the loop);
//   * the control block is replicated once per WARP (lane 0 runs the policy code of cuth_policy.cuh on its warp's
//     copy, __syncwarp): no block-wide barrier besides the ones inside the reductions.
// Same arithmetic per row as the flat kernels (spmv_row / fused_dir_spmv_row), same policy code, same stopping rule;
// FP64 and MIXED (difference form), M = diag A or I, steady and transient.  Selected automatically when the rows fit
// (cuth_api.cu), or with cuth_tuning_t.loop_mode = 3.  cuth_pcg_solve_batch launches one cluster per right-hand side.
#pragma once
#include <cooperative_groups.h>

#include "cuth_persistent.cuh"

namespace cuth {

constexpr int kClusterMaxCtas = 16;          // 8 = portable maximum, 16 = non-portable maximum on sm_100
constexpr int kClusterThreads = 1024;
constexpr int kClusterBytesPerRow = 136;     // r, z, x, mu, p, p2 (48) + 1/D0 (8) + 7 coefficients (56) + 6 neighbour words (24)
constexpr int kClusterFixedBytes = 16384;    // control blocks, reduction slots

struct ClusterSmem {
  // fixed part; the per-row arrays follow (carved in the kernel)
  Ctl ctl[kClusterThreads / 32];                        // one replica per warp
  double red[2][3][kClusterMaxCtas];                    // [parity][value][source CTA]
  double wsum[3][32];                                   // per-warp partial sums
  uint64_t bar[2];                                      // mbarriers of the all-reduce, used alternately
  Ctx ctx;                                              // the call's context: the policy code reads its options from
                                                        // here, not from global memory (every cluster barrier
                                                        // invalidates L1, an L2 round trip per field otherwise)
};
static_assert(sizeof(ClusterSmem) <= kClusterFixedBytes, "fixed part of the cluster kernel's shared memory");

// How the grid is dealt to the CTAs of the cluster: slabs along y or along z (whichever is longer), CTA c owning the
// slab [c*len/nc, (c+1)*len/nc).  Fewer rows then have a neighbour in another CTA than with a split of the linear index
// (cfg 1: 32 x 32 x 8 over 8 CTAs: y-slabs of 4 lines -- half a remote neighbour per row; z-slabs = single planes --
// two remote neighbours per row, and distributed shared memory moves only ~20 B per cycle and SM).
struct ClusterSplit { int axis_z; int len; };       // axis_z: 1 = slabs along z, 0 = along y
#ifdef __CUDACC__
__host__ __device__
#endif
inline ClusterSplit cluster_split(int64_t ny, int64_t nz) { return nz > ny ? ClusterSplit{1, (int)nz} : ClusterSplit{0, (int)ny}; }
inline int64_t cluster_rows_per_cta(int64_t nx, int64_t ny, int64_t nz, int nc) {
  const ClusterSplit sp = cluster_split(ny, nz);
  const int64_t thick = (sp.len + nc - 1) / nc;                 // thickest slab
  const int64_t r = nx * (sp.axis_z ? ny * thick : thick * nz);
  return (r + 31) / 32 * 32;
}
inline size_t cluster_smem_bytes(int64_t rows_per_cta) {
  return (size_t)kClusterFixedBytes + (size_t)kClusterBytesPerRow * (size_t)rows_per_cta;
}
inline bool cluster_fits(int64_t nx, int64_t ny, int64_t nz, int nc) {
  return cluster_smem_bytes(cluster_rows_per_cta(nx, ny, nz, nc)) <= (size_t)227 * 1024;
}

#ifdef __CUDACC__

// Sum of NV values over the whole cluster, identical in every thread of every CTA; also a cluster-wide barrier for every
// shared-memory write made before the call.
// NOT barrier.cluster: measured on B200 with 16 CTAs x 32 warps, an all-reduce built on cluster.sync() costs 2 700 -
// 3 500 cycles (every warp of every CTA takes part in the hardware barrier).  Here only NC lanes per CTA talk across
// CTAs: after the block-level sum, lane q of warp 0 sends the CTA's partial into CTA q's slot with st.async -- a remote
// store that carries its own completion signal: the 8 bytes are counted on CTA q's mbarrier (complete_tx) when they have
// landed -- and every thread waits on its OWN CTA's mbarrier, on which one local thread has announced the NC * NV * 8
// bytes of the phase (arrive.expect_tx).
//   * Round 2a used plain remote stores followed by mbarrier.arrive.release.cluster on the remote barrier: ptxas turns
//     that release into MEMBAR.ALL.GPU (+ CCTL.IVALL after the acquire.cluster wait), a GPU-scope fence twice per
//     iteration: cfg 1 in the register form 3.29 -> 2.64 us per iteration, in the shared-memory form 4.53 -> 3.97.
//   * Barrier property: a CTA sends only after its __syncthreads, i.e. after all its reads and writes of the phase (the
//     barrier instruction drains the CTA's shared-memory stores), and nobody passes before the bytes of every CTA have
//     landed; what the others then read remotely are ordinary shared-memory words written before that barrier.
//   * Two mbarriers, used alternately: a CTA can be one reduction ahead of another (never two -- to pass reduction n + 1
//     it needs every CTA's bytes of n + 1, sent after their wait of n), so its bytes for n + 1 must not count towards a
//     neighbour's still incomplete n.  `n` = index of the reduction: barrier n & 1, phase parity (n >> 1) & 1.
__device__ __forceinline__ uint32_t cl_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cl_mapa(uint32_t local_addr, unsigned rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cl_st_async(uint32_t remote_addr, double v, uint32_t remote_bar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(remote_addr), "d"(v),
               "r"(remote_bar) : "memory");
}
__device__ __forceinline__ void cl_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(cl_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cl_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "CL_WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra CL_WAIT_DONE;\n"
      "bra CL_WAIT_LOOP;\n"
      "CL_WAIT_DONE:\n"
      "}\n" ::"r"(cl_smem_u32(bar)), "r"(parity) : "memory");
}
// Once per kernel, by one thread, before the cluster-wide barrier that precedes the first reduction.
__device__ __forceinline__ void cluster_bars_init(ClusterSmem* sm) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(cl_smem_u32(&sm->bar[0])) : "memory");
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(cl_smem_u32(&sm->bar[1])) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// Butterfly over the low `W` lanes of each W-lane group (W a power of two <= 32): every lane ends with its group's sum.
template <int W>
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
  for (int o = W / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// FP64 adds and 64-bit shuffles are the narrow resources of this kernel (measured on B200: a dependent DADD ~25 cycles, a
// 5-level fp64 shuffle tree 210-260 cycles, and with 16 warps per SM the pipes themselves saturate), so the reduction is
// built to issue as few of them as possible:
//   1. in the warp, NV = 2: after the first exchange half the lanes carry value 0 and the other half value 1 -- one
//      butterfly for both values (10 shuffles + 5 adds per lane instead of 20 + 10);
//   2. across the warps of the CTA: warp k sums value k's NW partials, log2(NW) levels;
//   3. its lanes q < NC send the CTA's partial to CTA q (st.async, see above);
//   4. after the wait, the NC partials of value k are summed by the lanes of a 16-lane group, log2(NC) levels, and
//      broadcast -- NC loads and 2 NC adds per THREAD in round 2a.
// Every sum is a balanced tree of fixed shape: bit-reproducible, identical in all threads of all CTAs.
template <int NC, int NV, int NW = kClusterThreads / 32>      // NW: warps per CTA
__device__ __forceinline__ void cluster_allreduce(cg::cluster_group& cluster, ClusterSmem* sm, double (&v)[NV], int& n, long long* pr = nullptr) {
  static_assert(NV >= 1 && NV <= 3 && NC <= 16 && (NC & (NC - 1)) == 0 && (NW & (NW - 1)) == 0, "cluster_allreduce");
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int slot = n & 1;
#ifdef CUTH_CLUSTER_PROF
  long long q0 = clock64();
#define ARK(i) if (pr) { long long q1 = clock64(); pr[i] += q1 - q0; q0 = q1; }
#else
#define ARK(i)
#endif
  // ---- 1. the warp
  if (NV == 2) {
    const bool hi = (lane & 16) != 0;
    const double give = hi ? v[0] : v[1], keep = hi ? v[1] : v[0];
    const double w = group_sum<16>(keep + __shfl_xor_sync(0xffffffffu, give, 16));     // lanes 0-15: value 0, lanes 16-31: value 1
    if ((lane & 15) == 0) sm->wsum[lane >> 4][wid] = w;
  } else {
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = warp_sum(v[k]);
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < NV; ++k) sm->wsum[k][wid] = v[k];
    }
  }
  ARK(0)
  __syncthreads();
  ARK(1)
  // ---- 2, 3. the CTA, and out to the cluster
  if (wid < NV) {
    const unsigned me = cluster.block_rank();
    const double t = group_sum<(NW > NC ? NW : NC)>(lane < NW ? sm->wsum[wid][lane] : 0.0);   // lanes < NC must all hold the sum
    ARK(2)
    if (wid == 0 && lane == 0) cl_expect_tx(&sm->bar[slot], (uint32_t)(NC * NV * 8));
    if (lane < NC)
      cl_st_async(cl_mapa(cl_smem_u32(&sm->red[slot][wid][me]), (unsigned)lane), t,
                  cl_mapa(cl_smem_u32(&sm->bar[slot]), (unsigned)lane));                    // into CTA `lane`
  }
  ARK(3)
  cl_wait(&sm->bar[slot], (uint32_t)((n >> 1) & 1));
  ARK(4)
  // ---- 4. the cluster's sum
  if (NV <= 2) {
    const int k = NV == 2 ? lane >> 4 : 0, c = lane & 15;
    const double w = group_sum<NC>(c < NC ? sm->red[slot][k][c] : 0.0);
    v[0] = __shfl_sync(0xffffffffu, w, 0);
    if (NV == 2) v[1] = __shfl_sync(0xffffffffu, w, 16);
  } else {
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = __shfl_sync(0xffffffffu, group_sum<NC>(lane < NC ? sm->red[slot][k][lane] : 0.0), 0);
  }
  ARK(5)
  n += 1;
}

template <int NC>
__global__ void __launch_bounds__(kClusterThreads, 1) k_pcg_cluster(const Ctx* __restrict__ ctxp, Ctl* ctl_g, int rows_per_cta) {
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) unsigned char cl_raw[];
  ClusterSmem* sm = reinterpret_cast<ClusterSmem*>(cl_raw);
  const int R = rows_per_cta;
  // batched use (cuth_pcg_solve_batch): one cluster per right-hand side, each with its own context and control block
  ctxp += blockIdx.x / NC;
  ctl_g += blockIdx.x / NC;
  double* sr = reinterpret_cast<double*>(cl_raw + kClusterFixedBytes);
  double* sz = sr + R; double* sx = sz + R; double* smu = sx + R; double* sp0 = smu + R; double* sp1 = sp0 + R;
  double* sdi = sp1 + R;
  double* scf = sdi + R;                               // [7][R]: c0 (D0 or s), then the six off-diagonal coefficients
  uint32_t* snb = reinterpret_cast<uint32_t*>(scf + 7 * (size_t)R);   // [6][R]: owner CTA << 24 | index in the owner
  {
    const uint64_t* src = reinterpret_cast<const uint64_t*>(ctxp);
    uint64_t* dst = reinterpret_cast<uint64_t*>(&sm->ctx);
    for (int q = threadIdx.x; q < (int)(sizeof(Ctx) / 8); q += kClusterThreads) dst[q] = src[q];
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
  const size_t o_z = (size_t)kClusterFixedBytes + 8 * (size_t)R, o_x = o_z + 8 * (size_t)R,
               o_p0 = o_z + 24 * (size_t)R, o_p1 = o_z + 32 * (size_t)R;
  // element (owner, index) of the array at byte offset `off` of a CTA's block: a generic pointer into the distributed
  // shared memory of the cluster (mapa)
  auto remote = [&](uint32_t word, size_t off) -> const double* {
    return reinterpret_cast<const double*>(cluster.map_shared_rank(cl_raw + off, word >> 24)) + (word & 0xffffffu);
  };
  // ---- ownership: slabs along y or z
  const ClusterSplit sp = cluster_split(nyi, nzi);
  auto slab0 = [&](int q) { return (int)(((int64_t)q * sp.len) / NC); };
  auto owner_of = [&](int u) {                         // slab that holds coordinate u of the split axis
    int q = (int)(((int64_t)u * NC) / sp.len);
    while (q + 1 < NC && slab0(q + 1) <= u) ++q;
    while (q > 0 && slab0(q) > u) --q;
    return q;
  };
  const int s0 = slab0((int)me), s1 = slab0((int)me + 1);
  const int hy = sp.axis_z ? nyi : s1 - s0, hz = sp.axis_z ? s1 - s0 : nzi;
  const int my_rows = nxi * hy * hz;                   // <= R
  // local index of cell (x, y, z) in its owner q
  auto local_of = [&](int q, int x, int y, int z) {
    const int a0 = slab0(q), a1 = slab0(q + 1);
    return sp.axis_z ? x + nxi * (y + nyi * (z - a0)) : x + nxi * ((y - a0) + (a1 - a0) * z);
  };
  auto global_of = [&](int l) -> int64_t {             // global row of local row l of THIS CTA
    const int x = l % nxi, t = l / nxi, u = t % hy, v = t / hy;
    const int y = sp.axis_z ? u : u + s0, z = sp.axis_z ? v + s0 : v;
    return x + nx * (y + (int64_t)nyi * z);
  };

  // ---- load: coefficients of the stage, neighbour words, 1/D0, x0
  auto load_coefs = [&](bool early) {
    for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
      const int64_t i = global_of(l);
      double cf[7];
      const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = i + np < n, lo3 = i >= np;
      if (early) {          // fp32-stored off-diagonals promoted to fp64, difference form: c0 = s(z)
        cf[0] = A.s_layer[(unsigned)i / (unsigned)np];
        cf[1] = up1 ? (double)A.f1[i] : 0.0; cf[2] = lo1 ? (double)A.f1[i - 1] : 0.0;
        cf[3] = up2 ? (double)A.f2[i] : 0.0; cf[4] = lo2 ? (double)A.f2[i - nx] : 0.0;
        cf[5] = up3 ? (double)A.f3[i] : 0.0; cf[6] = lo3 ? (double)A.f3[i - np] : 0.0;
      } else {
        cf[0] = A.d0[i];
        cf[1] = up1 ? A.d1[i] : 0.0; cf[2] = lo1 ? A.d1[i - 1] : 0.0;
        cf[3] = up2 ? A.d2[i] : 0.0; cf[4] = lo2 ? A.d2[i - nx] : 0.0;
        cf[5] = up3 ? A.d3[i] : 0.0; cf[6] = lo3 ? A.d3[i - np] : 0.0;
      }
#pragma unroll
      for (int k = 0; k < 7; ++k) scf[(size_t)k * R + l] = cf[k];
    }
  };
  for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
    const int x = l % nxi, t = l / nxi, u = t % hy, v = t / hy;
    const int y = sp.axis_z ? u : u + s0, z = sp.axis_z ? v + s0 : v;
    const int64_t i = x + nx * (y + (int64_t)nyi * z);
    // neighbours in the order of Alg. 2 as the flat kernels add them: +1, -1, +nx, -nx, +nx*ny, -nx*ny.  The stored
    // structural zeros make the lateral wrap-around of the linear index harmless (coefficient 0); an absent neighbour
    // (or a wrapped one) is replaced by the row itself.
    const int dx[6] = {1, -1, 0, 0, 0, 0}, dy[6] = {0, 0, 1, -1, 0, 0}, dz[6] = {0, 0, 0, 0, 1, -1};
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const int xx = x + dx[k], yy = y + dy[k], zz = z + dz[k];
      uint32_t word = ((uint32_t)me << 24) | (uint32_t)l;
      if (xx >= 0 && xx < nxi && yy >= 0 && yy < nyi && zz >= 0 && zz < nzi) {
        const int q = owner_of(sp.axis_z ? zz : yy);
        word = ((uint32_t)q << 24) | (uint32_t)local_of(q, xx, yy, zz);
      }
      snb[(size_t)k * R + l] = word;
    }
    sdi[l] = jac ? A.dinv[i] : 1.0;
    sx[l] = c.x[i];
    sp0[l] = 0.0; sp1[l] = 0.0; sr[l] = 0.0; sz[l] = 0.0; smu[l] = 0.0;
  }
  if (lane == 0) *my = *ctl_g;                         // cleared by k_set_ctx
  if (threadIdx.x == 0) {
    cluster_bars_init(sm);
  }
  load_coefs(false);                                   // r0 = b - A1 x0 needs the fp64 operator
  cluster.sync();

  // y_l = (A v)_l for the stage in scf; v given by its array offset inside a CTA's block
  auto apply = [&](int l, size_t off, bool early) {
    const double vi = reinterpret_cast<const double*>(cl_raw + off)[l];
    double acc = scf[l] * vi;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const double vk = *remote(snb[(size_t)k * R + l], off);
      acc = fma(scf[(size_t)(k + 1) * R + l], early ? vk - vi : vk, acc);
    }
    return acc;
  };

  // ---- Alg. 1 lines 1-3
  {
    double acc[3] = {0.0, 0.0, 0.0};
    for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
      const double bi = c.b[global_of(l)];
      const double ri = bi - apply(l, o_x, false);
      const double zi = jac ? ri * sdi[l] : ri;
      sr[l] = ri; sz[l] = zi;
      acc[0] = fma(ri, zi, acc[0]); acc[1] = fma(ri, ri, acc[1]); acc[2] = fma(bi, bi, acc[2]);
    }
    cluster_allreduce<NC, 3>(cluster, sm, acc, parity);
    if (lane == 0) my->want_true = (int)policy_init(my, c, acc[0], acc[1], acc[2]);      // want_true reused as "go"
    __syncwarp();
  }
  bool go = my->want_true != 0;
  bool early = my->stage == 0;
  if (go && early) load_coefs(true);                   // rows are private to their thread: no barrier needed
  int pcur = 0;
#ifdef CUTH_CLUSTER_PROF
  long long tk[6] = {0, 0, 0, 0, 0, 0}, t0 = clock64(); unsigned long long g0; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g0)); int nit = 0;
#define CK(i) { long long t1 = clock64(); tk[i] += t1 - t0; t0 = t1; }
#else
#define CK(i)
#endif

  while (go) {
    // ---- AB: p' = z + beta p at the row and its six neighbours (z = M^-1 r was stored by its owner), mu = A p', p'.mu
    const double beta = my->beta;
    const size_t o_pold = pcur ? o_p1 : o_p0;
    double* pnew = pcur ? sp0 : sp1;
    double a1[1] = {0.0};
    for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
      const double pi = fma(beta, reinterpret_cast<const double*>(cl_raw + o_pold)[l], sz[l]);
      double acc = scf[l] * pi;
#pragma unroll
      for (int k = 0; k < 6; ++k) {
        const uint32_t wd = snb[(size_t)k * R + l];
        const double pk = fma(beta, *remote(wd, o_pold), *remote(wd, o_z));
        acc = fma(scf[(size_t)(k + 1) * R + l], early ? pk - pi : pk, acc);
      }
      pnew[l] = pi; smu[l] = acc;
      a1[0] = fma(pi, acc, a1[0]);
    }
    pcur ^= 1;
    CK(0)
    cluster_allreduce<NC, 1>(cluster, sm, a1, parity);
    CK(1)
    if (lane == 0) policy_after_spmv(my, a1[0], false);
    __syncwarp();
    CK(2)
    // ---- C: x, r, z, dots
    const double alpha = my->alpha;
    double a2[2] = {0.0, 0.0};
    for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
      sx[l] = fma(alpha, pnew[l], sx[l]);
      const double s0r = fma(-alpha, smu[l], sr[l]);
      const double z0 = jac ? s0r * sdi[l] : s0r;
      sr[l] = s0r; sz[l] = z0;
      a2[0] = fma(s0r, z0, a2[0]); a2[1] = fma(s0r, s0r, a2[1]);
    }
    CK(3)
    cluster_allreduce<NC, 2>(cluster, sm, a2, parity);
    CK(4)
    if (lane == 0) {
      unsigned g_, w_;
      policy_after_update(my, c, a2[0], a2[1], g_, w_);
      my->exiting = (int)g_;
    }
    __syncwarp();
    go = my->exiting != 0;
    CK(5)
#ifdef CUTH_CLUSTER_PROF
    ++nit;
#endif
    if (my->want_true) {
      // ---- D: true residual t = b - A1 x (x is complete: the all-reduce above was a cluster barrier)
      if (early) load_coefs(false);
      double a3[2] = {0.0, 0.0};
      for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
        const double ti = c.b[global_of(l)] - apply(l, o_x, false);
        const double di = ti - sr[l];
        smu[l] = ti;
        a3[0] = fma(ti, ti, a3[0]); a3[1] = fma(di, di, a3[1]);
      }
      cluster_allreduce<NC, 2>(cluster, sm, a3, parity);
      if (lane == 0) my->exiting = (int)policy_after_true(my, c, a3[0], a3[1]);
      __syncwarp();
      go = my->exiting != 0;
      const int mode = my->restart;
      early = my->stage == 0;
      if (go && early) load_coefs(true);               // still early: back to the fp32-stored coefficients
      if (go && mode) {
        // ---- E: r := t
        double a4[2] = {0.0, 0.0};
        for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) {
          const double ri = smu[l];
          const double zi = jac ? ri * sdi[l] : ri;
          sr[l] = ri; sz[l] = zi;
          a4[0] = fma(ri, zi, a4[0]); a4[1] = fma(ri, ri, a4[1]);
        }
        cluster_allreduce<NC, 2>(cluster, sm, a4, parity);
        if (lane == 0) policy_after_restart(my, c, mode, a4[0], a4[1]);
        __syncwarp();
      }
    }
  }
#ifdef CUTH_CLUSTER_PROF
  if (me == 0 && threadIdx.x == 0) { unsigned long long g1; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g1));
    printf("cluster prof NC=%d rows=%d its=%d ns/it=%.1f cyc/it: AB %.0f red1 %.0f pol1 %.0f C %.0f red2 %.0f pol2 %.0f\n", NC, my_rows, nit, (double)(g1 - g0) / nit,
           (double)tk[0] / nit, (double)tk[1] / nit, (double)tk[2] / nit, (double)tk[3] / nit, (double)tk[4] / nit, (double)tk[5] / nit); }
#endif
  // ---- epilogue: x back to the caller's buffer, result record
  if (!my->refused) {
    const bool zero = my->zero_rhs != 0;
    for (int l = threadIdx.x; l < my_rows; l += kClusterThreads) c.x[global_of(l)] = zero ? 0.0 : sx[l];
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
