// cuth_noalloc.cu -- ONE entry point for callers that cannot allocate: cuth_residual_noalloc.
//
// Some callers cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it),
// and every other reducing call of this library wants a caller-allocated workspace for its per-CTA partial sums.
// This file holds a variant of the true-residual kernel (k_true_resid: t = b - A1 x, ||t||^2, the
// quantity the stopping rule R-G7 is verified on) whose reduction scratch is a FILE-SCOPE device array of a fixed,
// modest size.  Consequences, all documented in include/cuth.h:
//   * a stated maximum problem size (kNoAllocMaxRows); larger grids are refused with CUTH_ERR_SIZE and a message;
//   * every GPU that loads the library holds the array (kNoAllocScratchBytes) until the process exits;
//   * all calls share the array and it keeps the last call's contents: the ticket is cleared at the start of every
//     call, every partial slot a call reads is written by that call first; two calls that OVERLAP on one GPU
//     (different streams) race on it -- serialise them.
// In host code the array's NAME is a host-side stand-in, not a device address: the address is fetched once per device,
// with that device current, by cudaGetSymbolAddress, and it is that pointer the kernel receives.
// Nothing here calls cudaMalloc, cudaFree or any allocating library routine.  No existing code path is changed.
#include <cmath>
#include <cstdio>
#include <mutex>
#include <string>
#include <unordered_map>

#include "cuth_internal.cuh"

namespace cuth {

constexpr int kNaThreads = 256;
constexpr int kNaRowsPerThread = 32;
constexpr int kNaRowsPerBlock = kNaThreads * kNaRowsPerThread;          // 8192 consecutive rows per CTA
constexpr int kNaMaxBlocks = 2048;                                      // partial slots per reduced value
constexpr int64_t kNoAllocMaxRows = (int64_t)kNaMaxBlocks * kNaRowsPerBlock;   // 2^24 = 16 777 216 rows (BASELINE cfg 3)
constexpr int kNaValues = 2;                                            // ||t||^2, ||b||^2
constexpr size_t kNoAllocScratchBytes = sizeof(double) * (kNaValues * kNaMaxBlocks + 32);   // 32 KB + one 256-B line

// The scratch: [0, 32) doubles = ticket line (word 0 used), then kNaValues x kNaMaxBlocks partial sums.
static __device__ __align__(256) double g_noalloc_scratch[kNaValues * kNaMaxBlocks + 32];

__device__ __forceinline__ double na_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Sums v[0..1] over the block; valid in thread 0.
__device__ __forceinline__ void na_block_sum(double (&v)[kNaValues], double* smem) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < kNaValues; ++k) v[k] = na_warp_sum(v[k]);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < kNaValues; ++k) smem[k * 32 + wid] = v[k];
  __syncthreads();
  if (wid == 0)
#pragma unroll
    for (int k = 0; k < kNaValues; ++k) v[k] = na_warp_sum(lane < kNaThreads / 32 ? smem[k * 32 + lane] : 0.0);
}

// t = b - A1 x on rows [blockIdx.x * 8192, ...), Alg. 2 read 0-based on the packed fp64 diagonals,
// same order of operations as spmv_row<OP_FP64>; per-CTA partials of ||t||^2 and ||b||^2 into the scratch; the last CTA
// to arrive (release-ordered ticket) adds them in a fixed order -- bit-reproducible -- and writes out[0..3].
__global__ void __launch_bounds__(kNaThreads) k_residual_noalloc(const double* __restrict__ d0, const double* __restrict__ d1,
                                                                const double* __restrict__ d2, const double* __restrict__ d3,
                                                                int64_t n, int64_t nx, int64_t np,
                                                                const double* __restrict__ b, const double* __restrict__ x,
                                                                double* __restrict__ t_out, double* scratch, double* out) {
  __shared__ double smem[kNaValues * 32];
  __shared__ int s_last;
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
  double* partials = scratch + 32;
  double acc[kNaValues] = {0.0, 0.0};
  const int64_t base = (int64_t)blockIdx.x * kNaRowsPerBlock;
#pragma unroll 4
  for (int k = 0; k < kNaRowsPerThread; ++k) {
    const int64_t i = base + (int64_t)k * kNaThreads + threadIdx.x;
    if (i < n) {
      const bool up1 = i + 1 < n, lo1 = i >= 1, up2 = i + nx < n, lo2 = i >= nx, up3 = i + np < n, lo3 = i >= np;
      const double a0 = d0[i];
      const double a1u = up1 ? d1[i] : 0.0, a1l = lo1 ? d1[i - 1] : 0.0;
      const double a2u = up2 ? d2[i] : 0.0, a2l = lo2 ? d2[i - nx] : 0.0;
      const double a3u = up3 ? d3[i] : 0.0, a3l = lo3 ? d3[i - np] : 0.0;
      const double v1u = up1 ? x[i + 1] : 0.0, v1l = lo1 ? x[i - 1] : 0.0;
      const double v2u = up2 ? x[i + nx] : 0.0, v2l = lo2 ? x[i - nx] : 0.0;
      const double v3u = up3 ? x[i + np] : 0.0, v3l = lo3 ? x[i - np] : 0.0;
      double ax = a0 * x[i];
      ax = fma(a1u, v1u, ax); ax = fma(a1l, v1l, ax);
      ax = fma(a2u, v2u, ax); ax = fma(a2l, v2l, ax);
      ax = fma(a3u, v3u, ax); ax = fma(a3l, v3l, ax);
      const double bi = b[i];
      const double ti = bi - ax;
      if (t_out) t_out[i] = ti;
      acc[0] = fma(ti, ti, acc[0]);
      acc[1] = fma(bi, bi, acc[1]);
    }
  }
  na_block_sum(acc, smem);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < kNaValues; ++k) __stcg(&partials[k * kNaMaxBlocks + blockIdx.x], acc[k]);
    unsigned int tk;
    asm volatile("atom.release.gpu.global.add.u32 %0, [%1], %2;" : "=r"(tk) : "l"(ticket), "r"(1u) : "memory");
    const int last = tk == gridDim.x - 1 ? 1 : 0;
    if (last) __threadfence();
    s_last = last;
  }
  __syncthreads();
  if (!s_last) return;
#pragma unroll
  for (int k = 0; k < kNaValues; ++k) {
    double a = 0.0;
    for (int c = threadIdx.x; c < (int)gridDim.x; c += kNaThreads) a += __ldcg(&partials[k * kNaMaxBlocks + c]);
    acc[k] = a;
  }
  na_block_sum(acc, smem);
  if (threadIdx.x == 0) {
    out[0] = acc[0];
    out[1] = acc[1];
    out[2] = acc[1] > 0.0 ? sqrt(acc[0] / acc[1]) : 0.0;
    out[3] = 0.0;
    *ticket = 0u;
  }
}

// Device address of the scratch, once per device (with that device current), under a mutex.
static std::mutex g_na_mu;
static std::unordered_map<int, double*> g_na_ptr;
static thread_local std::string g_na_err;

static cudaError_t noalloc_scratch(double** ptr) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lk(g_na_mu);
  auto it = g_na_ptr.find(dev);
  if (it == g_na_ptr.end()) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);      // NOT &g_noalloc_scratch: that is a host stand-in
    if (e != cudaSuccess || !p) return e != cudaSuccess ? e : cudaErrorInvalidSymbol;
    it = g_na_ptr.emplace(dev, p).first;
  }
  *ptr = it->second;
  return cudaSuccess;
}

}  // namespace cuth

using namespace cuth;

extern "C" {

int64_t cuth_noalloc_max_rows(void) { return kNoAllocMaxRows; }

const char* cuth_noalloc_last_error(void) { return g_na_err.c_str(); }

int cuth_residual_noalloc(const void* dia_D, const cuth_grid_t* grid, const double* b_D, const double* x_D,
                          double* t_D, double* out_D, void* stream) {
  g_na_err.clear();
  DiaLayout L;
  if (!grid) return CUTH_ERR_NULL;
  if (!make_layout(grid, &L)) { g_na_err = "cuth_residual_noalloc: nx, ny, nz must be >= 2 and N < 2^31"; return CUTH_ERR_DIMS; }
  if (L.n > kNoAllocMaxRows) {
    char buf[256];
    snprintf(buf, sizeof buf,
             "cuth_residual_noalloc: N = %lld rows exceeds the no-allocation path's maximum of %lld rows (its reduction "
             "scratch is a fixed %zu-byte device array); use a solver workspace instead",
             (long long)L.n, (long long)kNoAllocMaxRows, kNoAllocScratchBytes);
    g_na_err = buf;
    return CUTH_ERR_SIZE;
  }
  if (!dia_D || !b_D || !x_D || !out_D) return CUTH_ERR_NULL;
  if (((uintptr_t)dia_D & 15u) || ((uintptr_t)b_D & 7u) || ((uintptr_t)x_D & 7u) || ((uintptr_t)out_D & 7u) ||
      ((uintptr_t)t_D & 7u))
    return CUTH_ERR_ALIGN;
  if (t_D == x_D) return CUTH_ERR_VALUE;           // rows read their neighbours' x while others write t
  cudaStream_t st = (cudaStream_t)stream;
  double* scratch = nullptr;
  cudaError_t e = noalloc_scratch(&scratch);
  if (e == cudaSuccess) e = cudaMemsetAsync(scratch, 0, 256, st);          // the ticket line must start at zero
  if (e != cudaSuccess) {
    g_na_err = std::string("cuth_residual_noalloc: ") + cudaGetErrorString(e);
    cudaGetLastError();
    return CUTH_ERR_CUDA;
  }
  const char* base = (const char*)dia_D;
  const double* v = (const double*)(base + L.o_vals);
  const int blocks = (int)((L.n + kNaRowsPerBlock - 1) / kNaRowsPerBlock);
  k_residual_noalloc<<<blocks, kNaThreads, 0, st>>>(v + L.ptr[0], v + L.ptr[1], v + L.ptr[2], v + L.ptr[3], L.n, L.nx,
                                                    L.nxny, b_D, x_D, t_D, scratch, out_D);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    g_na_err = std::string("cuth_residual_noalloc: ") + cudaGetErrorString(e);
    return CUTH_ERR_CUDA;
  }
  return CUTH_OK;
}

}  // extern "C"
