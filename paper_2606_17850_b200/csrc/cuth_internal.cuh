// cuth_internal.cuh -- device-side structures and helpers shared by the cuth kernels.
// Product code (CUDA, sm_100a).  Shares nothing with oracle/.
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/cuth.h"

namespace cuth {

constexpr int kAlign = 256;            // byte alignment of every section of the matrix object / workspace
constexpr int kHeaderBytes = 512;
constexpr uint64_t kMagic = 0x4355544844494131ull;  // "CUTHDIA1"
constexpr int kMaxBlocks = 8192;       // upper bound on the grid of any reducing kernel
constexpr int kNumPartialSlots = 4;
constexpr int kMaxChebDegree = 64;    // partial-sum arrays (each kMaxBlocks doubles)
// 64-bit words of the matrix header (device memory; what the object IS is recorded in the object)
constexpr int kHdrMagic = 0, kHdrNx = 1, kHdrNy = 2, kHdrNz = 3, kHdrE = 4, kHdrTransient = 5, kHdrImported = 15,
              kHdrMixedOk = 16;

// Host-computed placement of the sections inside the caller's matrix buffer.
struct DiaLayout {
  int64_t nx, ny, nz, n, nxny, e;
  int64_t ptr[5], off[4];
  size_t o_layers;   // dz[nz] | s[nz] | cap[nz] | cvol[nz]   (fp64)
  size_t o_vals;     // fp64 [e]  packed D0|D1|D2|D3   (A1)
  size_t o_vals32;   // fp32 [e]  same packing          (A2)
  size_t o_dinv;     // fp64 [n]  1/D0
  size_t o_h16;      // fp16 3 x [n] (each 256-B aligned): off-diagonals D1, D2, D3 times a power-of-two scale (A3)
  size_t h16_stride; // bytes between the three fp16 arrays
  size_t o_f32a;     // fp32 3 x [n] (each 256-B aligned): the off-diagonals of A2 again, one array per diagonal, so
  size_t f32a_stride;//   that the pair (D_k[i], D_k[i+1]), i even, is one 8-byte load (packed D2, D3 start at odd elements)
  size_t o_f64a;     // fp64 3 x [n] (each 256-B aligned): the off-diagonals of A1 again, one array per diagonal with a zero
  size_t f64a_stride;//   tail: proper (nx, ny, nz) tensors for the TMA-staged K1 (packed D2, D3 start at odd elements, and a
                     //   tensor map needs a 16-byte aligned base)
  size_t o_dinv32;   // fp32 [n]: 1/D0 rounded to fp32 -- the Jacobi preconditioner of the EARLY stage of the fused path
                     //   ("fp32 storage where stable": M only has to be SPD; 8 B/row less in K1 and in K2)
  size_t bytes;
};

inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

inline bool make_layout(const cuth_grid_t* g, DiaLayout* L) {
  if (!g || g->nx < 2 || g->ny < 2 || g->nz < 2) return false;
  if (g->nx > (1ll << 31) / g->ny || g->nx * g->ny > (1ll << 31) / g->nz) return false;  // N < 2^31
  L->nx = g->nx; L->ny = g->ny; L->nz = g->nz;
  L->nxny = g->nx * g->ny;
  L->n = L->nxny * g->nz;
  L->off[0] = 0; L->off[1] = 1; L->off[2] = g->nx; L->off[3] = L->nxny;
  L->ptr[0] = 0;
  for (int k = 0; k < 4; ++k) L->ptr[k + 1] = L->ptr[k] + (L->n - L->off[k]);
  L->e = L->ptr[4];
  size_t o = kHeaderBytes;
  L->o_layers = o; o = align_up(o + (4 * (size_t)g->nz + 4) * sizeof(double));   // + absmax bits, scale, 1/scale, spare
  L->o_vals = o;   o = align_up(o + sizeof(double) * (size_t)L->e);
  L->o_vals32 = o; o = align_up(o + sizeof(float) * (size_t)L->e);
  L->o_dinv = o;   o = align_up(o + sizeof(double) * (size_t)L->n);
  L->h16_stride = align_up(sizeof(__half) * (size_t)L->n);
  L->o_h16 = o;    o = o + 3 * L->h16_stride;
  L->f32a_stride = align_up(sizeof(float) * (size_t)L->n);
  L->o_f32a = o;   o = o + 3 * L->f32a_stride;
  L->f64a_stride = align_up(sizeof(double) * (size_t)L->n);
  L->o_f64a = o;   o = o + 3 * L->f64a_stride;
  L->o_dinv32 = o; o = align_up(o + sizeof(float) * (size_t)L->n);
  L->bytes = o;
  return true;
}

// Device view of the matrix handed to kernels by value.
struct DiaDev {
  const double* d0; const double* d1; const double* d2; const double* d3;   // fp64 diagonals (A1)
  const float* f0;                                                          // fp32 main diagonal (A2), ablation only
  const float* f1; const float* f2; const float* f3;                        // fp32 off-diagonals (A2): the aligned
                                                                            // per-diagonal copies, [n] each, zero tail
  const __half* h1; const __half* h2; const __half* h3;                     // fp16 off-diagonals x scale (A3)
  const double* h_scale;    // [0] absmax bits, [1] scale (power of two), [2] 1/scale
  const double* dinv;       // 1/D0
  const float* dinv32;      // fp32(1/D0): M^-1 of the early stage on the fused path
  const double* s_layer;    // exact row sums per layer: h dx dy [top] + C V / dt
  const double* cap_layer;  // C V / dt per layer (0 when steady)
  const unsigned long long* hdr;   // the object's header (kHdr* words)
  int64_t n, nx, nxny;
  int32_t ny, nz;
  int32_t zmarch, x2;       // zmarch 1: march in z per thread (plane neighbours in registers), 0: flat 1-D
                            // streaming; x2 1: two x-adjacent columns per thread (nx even), 16-byte vector loads
};

// Pointers and options of one solve; lives at the start of the workspace, written per call.
struct Ctx {
  DiaDev A;
  const double* b;
  double* x;
  double* r;
  double* p;
  double* p2;      // second direction buffer (fused path ping-pongs p between p and p2)
  double* mu;
  cuth_result_t* result;
  double rtol;
  double soft_drift2;   // soft restart allowed while ||t - r||^2 <= soft_drift2 * ||t||^2
  int32_t precision, max_iters, period, jacobi;
  int32_t soft_restart, cheb;     // cheb: degree k of the Chebyshev polynomial preconditioner, 0 = off
  int32_t persist_fuse;           // persistent kernel: phases A and B in one (p' recomputed at the six neighbours)
  int32_t early_op;               // operator of the early stage: 1 = difference form (R-F3), 2 = A2 in standard form (ablation)
  int32_t transient_call;         // 1: cuth_transient_step (the matrix object must be a transient one)
  int32_t k1_split;               // graph loop on thin stacks (nz < 12): the TMA-staged K1 serves the early stage only, the
                                  // two-column LDG K1 the late stage; each returns at once in the other's stage
  // Chebyshev preconditioner (Alg. 3): z = q(A) r.  cz: z (fp64) handed to the outer
  // loop; cd[4]: partial-sum buffers Z (two are live at any time; the fused two-pass kernel writes the other
  // two); crc: fp32 copy of r (MIXED only).  Element type T = double in FP64 mode, float in MIXED mode;
  // cd[0], cd[1] are sized for double, cd[2], cd[3] for float (the two-pass kernel is fp32 only).
  double* cz; void* cd[4]; void* crc;
  double cheb_inv_theta;
  double cheb_c1[kMaxChebDegree], cheb_c2[kMaxChebDegree];   // d_{i+1} = c1[i] d_i + c2[i] r_c
};

// Scalars of the iteration; device resident, written only by "last block" epilogues.
struct Ctl {
  double rho, pAp, alpha, beta, rr, bb, tol2, sw2;
  double tt, dd, tt_prev, rr_prev_eval;
  double xalpha;   // pending x += xalpha * p (fused path defers Alg. 1 line 8 by one kernel)
  int32_t it, stage, status, want_true, restart, exiting, promotions, evals, since_eval;
  int32_t switch_reason, switch_it, conv_rec, zero_rhs, no_graph, pcur, beta_zero, switch_mask;
  int32_t hard_restarts, soft_restarts, refused;
  int32_t xnow;    // fused path: K2 of this iteration applies x += alpha p itself (an evaluation is certain to follow)
  int32_t halt;    // graph loop with an unrolled body: the remaining K1 / K2 launches of this pass are no-ops
                   // (the loop must stop, or the true-residual branch at the end of the body must run first)
  unsigned int ticket[8];
};

struct Workspace {
  Ctx* ctx; Ctl* ctl; double* partials; double* r; double* p; double* p2; double* mu; double* b;
  double* cz; double* cd0; double* cd1; double* crc; float* cd2; float* cd3;
  size_t bytes;
};

inline Workspace carve_workspace(void* base, int64_t n, bool with_b, bool with_cheb = false) {
  Workspace w;
  char* c = (char*)base;
  size_t o = 0;
  w.ctx = (Ctx*)(c + o); o = align_up(o + sizeof(Ctx));
  w.ctl = (Ctl*)(c + o); o = align_up(o + sizeof(Ctl));
  w.partials = (double*)(c + o); o = align_up(o + sizeof(double) * kMaxBlocks * kNumPartialSlots);
  w.r = (double*)(c + o); o = align_up(o + sizeof(double) * (size_t)n);
  w.p = (double*)(c + o); o = align_up(o + sizeof(double) * (size_t)n);
  w.p2 = (double*)(c + o); o = align_up(o + sizeof(double) * (size_t)n);
  w.mu = (double*)(c + o); o = align_up(o + sizeof(double) * (size_t)n);
  w.b = nullptr;
  if (with_b) { w.b = (double*)(c + o); o = align_up(o + sizeof(double) * (size_t)n); }
  w.cz = w.cd0 = w.cd1 = w.crc = nullptr;
  w.cd2 = w.cd3 = nullptr;
  if (with_cheb) {
    double** v[4] = {&w.cz, &w.cd0, &w.cd1, &w.crc};
    for (int k = 0; k < 4; ++k) { *v[k] = (double*)(c + o); o = align_up(o + sizeof(double) * (size_t)n); }
    w.cd2 = (float*)(c + o); o = align_up(o + sizeof(float) * (size_t)n);
    w.cd3 = (float*)(c + o); o = align_up(o + sizeof(float) * (size_t)n);
  }
  w.bytes = o;
  return w;
}

#ifdef __CUDACC__
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sum of NV values over the block (blockDim.x multiple of 32, <= 1024); result valid in thread 0.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* smem /* >= NV*32 */) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = warp_sum(v[k]);
  __syncthreads();
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) smem[k * 32 + wid] = v[k];
  }
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      double t = lane < nw ? smem[k * 32 + lane] : 0.0;
      v[k] = warp_sum(t);
    }
  }
}

// Grid-wide deterministic reduction: every block deposits NV partials, the last block to arrive
// (atomic ticket) sums them in a fixed order.  Returns true in ALL threads of that last block,
// with the totals valid in thread 0 only.
template <int NV>
__device__ __forceinline__ bool grid_sum_last_block(double (&v)[NV], double* partials, unsigned int* ticket,
                                                    double* smem, int* s_flag) {
  block_sum<NV>(v, smem);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) __stcg(&partials[k * kMaxBlocks + blockIdx.x], v[k]);
    // Release-only ticket: orders the partial stores before the increment WITHOUT the L1 invalidation
    // (CCTL.IVALL) that __threadfence() costs every CTA -- the in-plane stencil neighbours live in L1.
    unsigned int t;
    asm volatile("atom.release.gpu.global.add.u32 %0, [%1], %2;" : "=r"(t) : "l"(ticket), "r"(1u) : "memory");
    const int last = (t == gridDim.x - 1) ? 1 : 0;
    if (last) __threadfence();     // acquire side, paid by the single last CTA; partials are read with ld.cg
    *s_flag = last;
  }
  __syncthreads();
  if (!*s_flag) return false;
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    double a = 0.0;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) a += __ldcg(&partials[k * kMaxBlocks + b]);
    v[k] = a;
  }
  block_sum<NV>(v, smem);
  if (threadIdx.x == 0) *ticket = 0u;
  return true;
}
#endif  // __CUDACC__

}  // namespace cuth
