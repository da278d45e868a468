// cuth_build.cu -- condensed-DIA ("Quad-Diag") builder kernel: hot-path step a0.
// One thread per cell evaluates eq. (4)/(5) and writes the main and the
// three upper diagonals, the fp32 copy A2, and 1/D0.  Every fp64 operation is an explicit
// round-to-nearest intrinsic (no FMA contraction), in the order stated in DESIGN.md §4, so the
// stored values can be compared bit for bit with an independently assembled matrix.
#include <cmath>
#include <cstring>
#include <vector>

#include "cuth_internal.cuh"

namespace cuth {

struct BuildArgs {
  int64_t nx, ny, nz, n, nxny;
  double dx, dy, h_top, dt;
  const double* dz;      // device [nz] (inside the matrix object)
  const double* cvol;    // device [nz] or nullptr (inside the matrix object: cap staging area)
  const double* kappa;   // device, nz or n values
  int per_layer, transient;
  double* d0; double* d1; double* d2; double* d3;
  float* f0; float* f1; float* f2; float* f3;
  double* dinv;
};

__device__ __forceinline__ double series2(double area, double la, double ka, double lb, double kb) {
  // area / ( la/(2 ka) + lb/(2 kb) ): two half cells in series between neighbouring cell centres
  return __ddiv_rn(area, __dadd_rn(__ddiv_rn(la, __dmul_rn(2.0, ka)), __ddiv_rn(lb, __dmul_rn(2.0, kb))));
}

__global__ void __launch_bounds__(256) build_dia_kernel(BuildArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    const int64_t z = i / a.nxny;
    const int64_t rem = i - z * a.nxny;
    const int64_t y = rem / a.nx;
    const int64_t x = rem - y * a.nx;
    const double dzz = a.dz[z];
    auto kap = [&](int64_t j, int64_t zz) { return a.per_layer ? a.kappa[zz] : a.kappa[j]; };
    const double k0 = kap(i, z);
    const double ayz = __dmul_rn(a.dy, dzz);   // face area normal to x
    const double axz = __dmul_rn(a.dx, dzz);   // face area normal to y
    const double axy = __dmul_rn(a.dx, a.dy);  // face area normal to z
    double diag = 0.0;
    // lower neighbours first (-z, -y, -x), a = the lower-index cell
    if (z > 0) diag = __dadd_rn(diag, series2(axy, a.dz[z - 1], kap(i - a.nxny, z - 1), dzz, k0));
    if (y > 0) diag = __dadd_rn(diag, series2(axz, a.dy, kap(i - a.nx, z), a.dy, k0));
    if (x > 0) diag = __dadd_rn(diag, series2(ayz, a.dx, kap(i - 1, z), a.dx, k0));
    double gx = 0.0, gy = 0.0, gz = 0.0;
    const bool hx = x + 1 < a.nx, hy = y + 1 < a.ny, hz = z + 1 < a.nz;
    if (hx) { gx = series2(ayz, a.dx, k0, a.dx, kap(i + 1, z)); diag = __dadd_rn(diag, gx); }
    if (hy) { gy = series2(axz, a.dy, k0, a.dy, kap(i + a.nx, z)); diag = __dadd_rn(diag, gy); }
    if (hz) { gz = series2(axy, dzz, k0, a.dz[z + 1], kap(i + a.nxny, z + 1)); diag = __dadd_rn(diag, gz); }
    if (z == a.nz - 1) diag = __dadd_rn(diag, __dmul_rn(a.h_top, axy));                      // Robin top
    if (a.transient) diag = __dadd_rn(diag, __ddiv_rn(__dmul_rn(a.cvol[z], __dmul_rn(axy, dzz)), a.dt));
    a.d0[i] = diag;
    a.f0[i] = __double2float_rn(diag);
    a.dinv[i] = __ddiv_rn(1.0, diag);
    if (i + 1 < a.n) { const double v = hx ? -gx : 0.0; a.d1[i] = v; a.f1[i] = __double2float_rn(v); }
    if (i + a.nx < a.n) { const double v = hy ? -gy : 0.0; a.d2[i] = v; a.f2[i] = __double2float_rn(v); }
    if (hz) { a.d3[i] = -gz; a.f3[i] = __double2float_rn(-gz); }
  }
}

// A3: half-precision copy of the off-diagonals.  The entries of these matrices are
// 1e-8..1 W/K, far below fp16's normal range, so they are stored times a power of two S chosen from the
// largest |entry| (S * max in (2^13, 2^14]); the kernels multiply the accumulated sum by 1/S once.
__global__ void __launch_bounds__(256) k_offdiag_absmax(const double* __restrict__ v, int64_t count, double* slot) {
  double m = 0.0;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += stride) m = fmax(m, fabs(v[i]));
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax((unsigned long long*)slot, (unsigned long long)__double_as_longlong(m));
}

__global__ void k_h16_scale(double* slot) {
  const double m = __longlong_as_double((long long)((unsigned long long*)slot)[0]);
  int e = 0;
  if (m > 0.0) { frexp(m, &e); }                 // m = f * 2^e, f in [0.5, 1)
  const double scale = ldexp(1.0, 14 - e);       // S * m in [2^13, 2^14)
  slot[1] = scale;
  slot[2] = 1.0 / scale;
}

__global__ void __launch_bounds__(256) k_make_h16(BuildArgs a, const double* slot, __half* h1, __half* h2, __half* h3) {
  const double scale = slot[1];
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    h1[i] = __double2half(i + 1 < a.n ? a.d1[i] * scale : 0.0);
    h2[i] = __double2half(i + a.nx < a.n ? a.d2[i] * scale : 0.0);
    h3[i] = __double2half(i + a.nxny < a.n ? a.d3[i] * scale : 0.0);
  }
}

// The off-diagonals of A2 once more, one 256-B aligned array of n floats per diagonal (zero beyond the
// diagonal's length): what the solver kernels read.  The packed fp32 copy stays what cuth_dia_view shows.
// ... and the same for the fp64 off-diagonals of A1 (e1..e3): the operands of the TMA-staged K1 (cuth_fused_tma.cuh).
__global__ void __launch_bounds__(256) k_make_f32a(BuildArgs a, float* g1, float* g2, float* g3, double* e1, double* e2,
                                                   double* e3, float* dinv32) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    const bool h1 = i + 1 < a.n, h2 = i + a.nx < a.n, h3 = i + a.nxny < a.n;
    g1[i] = h1 ? a.f1[i] : 0.f;
    g2[i] = h2 ? a.f2[i] : 0.f;
    g3[i] = h3 ? a.f3[i] : 0.f;
    e1[i] = h1 ? a.d1[i] : 0.0;
    e2[i] = h2 ? a.d2[i] : 0.0;
    e3[i] = h3 ? a.d3[i] : 0.0;
    dinv32[i] = __double2float_rn(a.dinv[i]);      // fp32(1/D0): the early-stage Jacobi preconditioner of the fused path
  }
}

// Small host arrays (header, per-layer tables) reach the matrix object as KERNEL ARGUMENTS, 64 words per launch:
// no pageable cudaMemcpyAsync (which blocks the host and cannot be stream-captured), no pinned staging buffer to
// keep alive -- cuth_build_dia is asynchronous and capturable like every other call.
struct WordChunk { unsigned long long w[64]; };
__global__ void k_write_words(unsigned long long* dst, WordChunk c, int count) {
  if ((int)threadIdx.x < count) dst[threadIdx.x] = c.w[threadIdx.x];
}
static cudaError_t write_words(void* dst, const void* src_H, size_t nwords, cudaStream_t st) {
  const unsigned long long* src = (const unsigned long long*)src_H;
  for (size_t o = 0; o < nwords; o += 64) {
    WordChunk c;
    const int cnt = (int)(nwords - o < 64 ? nwords - o : 64);
    memcpy(c.w, src + o, sizeof(unsigned long long) * (size_t)cnt);
    k_write_words<<<1, 64, 0, st>>>((unsigned long long*)dst + o, c, cnt);
  }
  return cudaGetLastError();
}

// Host side: fills the per-layer arrays, launches the kernel.  Called from cuth_api.cu.
int launch_build(const cuth_grid_t* g, const DiaLayout& L, void* dia_D, cudaStream_t st, cudaError_t* err) {
  char* base = (char*)dia_D;
  const int nz = (int)g->nz;
  const bool transient = g->cvol_H != nullptr && g->dt > 0.0;
  // per-layer arrays inside the matrix object: dz | s | cap | cvol
  std::vector<double> hv(4 * (size_t)nz + 4);
  double* h = hv.data();
  for (int k = 0; k < 4; ++k) h[4 * nz + k] = 0.0;
  for (int z = 0; z < nz; ++z) {
    const double axy = g->dx * g->dy;
    const double cap = transient ? g->cvol_H[z] * (axy * g->dz_H[z]) / g->dt : 0.0;
    h[z] = g->dz_H[z];
    h[nz + z] = (z == nz - 1 ? g->h_top * axy : 0.0) + cap;
    h[2 * nz + z] = cap;
    h[3 * nz + z] = transient ? g->cvol_H[z] : 0.0;
  }
  // header
  unsigned long long hdr[kHeaderBytes / 8] = {0};
  hdr[0] = kMagic; hdr[1] = (unsigned long long)g->nx; hdr[2] = (unsigned long long)g->ny;
  hdr[3] = (unsigned long long)g->nz; hdr[4] = (unsigned long long)L.e; hdr[5] = transient ? 1ull : 0ull;
  for (int k = 0; k < 5; ++k) hdr[6 + k] = (unsigned long long)L.ptr[k];
  for (int k = 0; k < 4; ++k) hdr[11 + k] = (unsigned long long)L.off[k];
  hdr[kHdrImported] = 0ull; hdr[kHdrMixedOk] = 1ull;
  cudaError_t e = write_words(base, hdr, kHeaderBytes / 8, st);
  if (e == cudaSuccess) e = write_words(base + L.o_layers, h, 4 * (size_t)nz + 4, st);
  if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
  BuildArgs a;
  a.nx = L.nx; a.ny = L.ny; a.nz = L.nz; a.n = L.n; a.nxny = L.nxny;
  a.dx = g->dx; a.dy = g->dy; a.h_top = g->h_top; a.dt = g->dt;
  a.dz = (const double*)(base + L.o_layers);
  a.cvol = (const double*)(base + L.o_layers) + 3 * nz;
  a.kappa = g->kappa_D;
  a.per_layer = g->kappa_is_per_layer ? 1 : 0;
  a.transient = transient ? 1 : 0;
  double* v = (double*)(base + L.o_vals);
  float* f = (float*)(base + L.o_vals32);
  a.d0 = v + L.ptr[0]; a.d1 = v + L.ptr[1]; a.d2 = v + L.ptr[2]; a.d3 = v + L.ptr[3];
  a.f0 = f + L.ptr[0]; a.f1 = f + L.ptr[1]; a.f2 = f + L.ptr[2]; a.f3 = f + L.ptr[3];
  a.dinv = (double*)(base + L.o_dinv);
  int64_t blocks = (L.n + 255) / 256;
  if (blocks > 148 * 64) blocks = 148 * 64;
  build_dia_kernel<<<(unsigned)blocks, 256, 0, st>>>(a);
  double* slot = (double*)(base + L.o_layers) + 4 * nz;
  k_offdiag_absmax<<<(unsigned)blocks, 256, 0, st>>>(a.d1, L.e - L.n, slot);     // D1|D2|D3 are contiguous
  k_h16_scale<<<1, 1, 0, st>>>(slot);
  k_make_h16<<<(unsigned)blocks, 256, 0, st>>>(a, slot, (__half*)(base + L.o_h16),
                                               (__half*)(base + L.o_h16 + L.h16_stride),
                                               (__half*)(base + L.o_h16 + 2 * L.h16_stride));
  k_make_f32a<<<(unsigned)blocks, 256, 0, st>>>(a, (float*)(base + L.o_f32a), (float*)(base + L.o_f32a + L.f32a_stride),
                                                (float*)(base + L.o_f32a + 2 * L.f32a_stride), (double*)(base + L.o_f64a),
                                                (double*)(base + L.o_f64a + L.f64a_stride),
                                                (double*)(base + L.o_f64a + 2 * L.f64a_stride), (float*)(base + L.o_dinv32));
  e = cudaGetLastError();
  if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
  return CUTH_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Importer ("CSR / COO import", PAPER.md:430 -- the paper's matrices arrive as sparse matrices
// from 3D-ICE and are then "decomposed and stored as a set of diagonal vectors").  A CSR matrix
// whose structure is the 7-point stencil of an nx x ny x nz box is checked and condensed into the same matrix
// object cuth_build_dia writes: the four upper diagonals are COPIED (bit-exact), the lower triangle is only
// compared with its mirror.
struct ImportArgs {
  int64_t n, nx, ny, nxny;
  int32_t nz;
  const int64_t* rowptr; const int32_t* col; const double* val;
  const int32_t* coo_row; int64_t nnz; unsigned int* seen;   // COO input: row index per entry; seen[n]: slot bits per row
  double* d0; double* d1; double* d2; double* d3;
  unsigned long long* cnt;     // [0] off-stencil, [1] asymmetric, [2] bad diagonal, [3] duplicates, [4] positive off-diagonals
  unsigned long long* rs_min;  // [nz] order-preserving keys of the per-layer min / max row sum and min D0
  unsigned long long* rs_max;
  unsigned long long* d0_min;
};

__device__ __forceinline__ unsigned long long ordered_key(double v) {   // monotone map double -> uint64
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}

// Pass 0: is rowptr a row pointer at all?  A malformed one would send the passes below out of bounds through col / val
// (or into a very long loop), so nothing else is read until this count is zero.
__global__ void __launch_bounds__(256) k_import_check_rowptr(const int64_t* __restrict__ rowptr, int64_t n, int64_t nnz,
                                                            unsigned long long* bad_out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned long long bad = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const int64_t lo = rowptr[i], hi = rowptr[i + 1];
    if (lo < 0 || hi < lo || hi - lo > 4096 || (i == 0 && lo != 0) || (nnz >= 0 && hi > nnz)) ++bad;
  }
  if (bad) atomicAdd(bad_out, bad);
}

// Pass 1, one thread per row: the row's own diagonal and upper entries go to their slots (a missing entry is
// +0.0, which is also what the builder stores where the +x / +y neighbour does not exist).
__global__ void __launch_bounds__(256) k_import_upper(ImportArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned long long off_st = 0, bad = 0, dup = 0, pos = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    const int64_t rem = i % a.nxny;
    const int64_t x = rem % a.nx, y = rem / a.nx;
    double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0;
    unsigned seen = 0;
    for (int64_t q = a.rowptr[i]; q < a.rowptr[i + 1]; ++q) {
      const int64_t cq = (int64_t)a.col[q];
      const int64_t c = cq - i;
      const double v = a.val[q];
      int slot = -1;
      bool legal = cq >= 0 && cq < a.n;
      if (c == 0) slot = 0;
      else if (c == 1) { slot = 1; legal = legal && x + 1 < a.nx; }
      else if (c == a.nx) { slot = 2; legal = legal && y + 1 < a.ny; }
      else if (c == a.nxny) slot = 3;
      else if (c == -1) { slot = 4; legal = legal && x > 0; }
      else if (c == -a.nx) { slot = 5; legal = legal && y > 0; }
      else if (c == -a.nxny) slot = 6;
      if (slot < 0 || !legal) { if (v != 0.0) ++off_st; continue; }   // explicit zeros off the stencil are ignored
      if (seen & (1u << slot)) { ++dup; continue; }
      seen |= 1u << slot;
      if (slot == 0) v0 = v; else if (slot == 1) v1 = v; else if (slot == 2) v2 = v; else if (slot == 3) v3 = v;
      if (slot != 0 && v > 0.0) ++pos;
    }
    if (!(seen & 1u) || !(v0 > 0.0) || isinf(v0)) ++bad;
    a.d0[i] = v0;
    if (i + 1 < a.n) a.d1[i] = v1;
    if (i + a.nx < a.n) a.d2[i] = v2;
    if (i + a.nxny < a.n) a.d3[i] = v3;
  }
  if (off_st) atomicAdd(&a.cnt[0], off_st);
  if (bad) atomicAdd(&a.cnt[2], bad);
  if (dup) atomicAdd(&a.cnt[3], dup);
  if (pos) atomicAdd(&a.cnt[4], pos);
}

// Row sum D0 + the six off-diagonal entries of row i in the fixed order -z, -y, -x, +x, +y, +z (m1..m3: the stored
// mirrors of the lower entries), folded into the per-layer min / max of the row sums and min of D0.
__device__ __forceinline__ void rowsum_minmax(const ImportArgs& a, int64_t i, double m1, double m2, double m3) {
  const double d = a.d0[i];
  double rs = d;
  rs = __dadd_rn(rs, m3); rs = __dadd_rn(rs, m2); rs = __dadd_rn(rs, m1);
  if (i + 1 < a.n) rs = __dadd_rn(rs, a.d1[i]);
  if (i + a.nx < a.n) rs = __dadd_rn(rs, a.d2[i]);
  if (i + a.nxny < a.n) rs = __dadd_rn(rs, a.d3[i]);
  const int64_t z = i / a.nxny;
  // a full warp inside one layer (the common case) reduces by shuffle: one atomic per warp and quantity
  unsigned long long kmin = ordered_key(rs), kmax = kmin, kd = ordered_key(d);
  const unsigned mask = __activemask();
  bool uniform = false;
  if (mask == 0xffffffffu) {
    const int64_t z0 = __shfl_sync(mask, z, 0);
    uniform = __all_sync(mask, z == z0);
    if (uniform) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long t1 = __shfl_xor_sync(mask, kmin, o), t2 = __shfl_xor_sync(mask, kmax, o),
                                 t3 = __shfl_xor_sync(mask, kd, o);
        kmin = t1 < kmin ? t1 : kmin; kmax = t2 > kmax ? t2 : kmax; kd = t3 < kd ? t3 : kd;
      }
    }
  }
  if (!uniform || (threadIdx.x & 31) == 0) {
    atomicMin(&a.rs_min[z], kmin); atomicMax(&a.rs_max[z], kmax); atomicMin(&a.d0_min[z], kd);
  }
}

// Pass 2, one thread per row: every lower entry must equal the stored mirror (absent == 0), and the row sum
// D0 + sum of the six off-diagonal entries (fixed order -z, -y, -x, +x, +y, +z) feeds the per-layer min / max.
__global__ void __launch_bounds__(256) k_import_lower(ImportArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned long long asym = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    double l1 = 0.0, l2 = 0.0, l3 = 0.0;
    unsigned seen = 0;
    const int64_t rem = i % a.nxny;
    const bool has_xm = rem % a.nx > 0, has_ym = rem / a.nx > 0;     // edge-crossing entries were counted in pass 1
    for (int64_t q = a.rowptr[i]; q < a.rowptr[i + 1]; ++q) {
      const int64_t c = (int64_t)a.col[q] - i;
      const double v = a.val[q];
      if (c == -1 && has_xm && !(seen & 1u)) { l1 = v; seen |= 1u; }
      else if (c == -a.nx && has_ym && !(seen & 2u)) { l2 = v; seen |= 2u; }
      else if (c == -a.nxny && !(seen & 4u)) { l3 = v; seen |= 4u; }
    }
    const double m1 = i >= 1 ? a.d1[i - 1] : 0.0;
    const double m2 = i >= a.nx ? a.d2[i - a.nx] : 0.0;
    const double m3 = i >= a.nxny ? a.d3[i - a.nxny] : 0.0;
    if (!(l1 == m1) || !(l2 == m2) || !(l3 == m3)) ++asym;
    rowsum_minmax(a, i, m1, m2, m3);
  }
  if (asym) atomicAdd(&a.cnt[1], asym);
}

// ---- COO input (SURVEY.md §8(f) "CSR / COO import"): the same checks with one thread per ENTRY.
// seen[i] bit s (s = 0 diagonal, 1..3 upper +1 / +nx / +nx*ny, 4..6 lower) = an on-stencil entry of row i was met in
// slot s; bit 8 = a lower entry of row i differs from its mirror.
__device__ __forceinline__ int coo_slot(const ImportArgs& a, int64_t i, int64_t j, bool* legal) {
  *legal = i >= 0 && i < a.n && j >= 0 && j < a.n;
  if (!*legal) return -1;
  const int64_t c = j - i, rem = i % a.nxny, x = rem % a.nx, y = rem / a.nx;
  if (c == 0) return 0;
  if (c == 1) { *legal = x + 1 < a.nx; return 1; }
  if (c == a.nx) { *legal = y + 1 < a.ny; return 2; }
  if (c == a.nxny) return 3;
  if (c == -1) { *legal = x > 0; return 4; }
  if (c == -a.nx) { *legal = y > 0; return 5; }
  if (c == -a.nxny) return 6;
  return -1;
}

__global__ void __launch_bounds__(256) k_coo_scatter(ImportArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned long long off_st = 0, dup = 0, pos = 0;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < a.nnz; q += stride) {
    const int64_t i = a.coo_row[q], j = a.col[q];
    const double v = a.val[q];
    bool legal;
    const int slot = coo_slot(a, i, j, &legal);
    if (slot < 0 || !legal) { if (v != 0.0) ++off_st; continue; }
    const unsigned old = atomicOr(&a.seen[i], 1u << slot);
    if (old & (1u << slot)) { ++dup; continue; }
    if (slot == 0) a.d0[i] = v; else if (slot == 1) a.d1[i] = v; else if (slot == 2) a.d2[i] = v; else if (slot == 3) a.d3[i] = v;
    if (slot != 0 && v > 0.0) ++pos;
  }
  if (off_st) atomicAdd(&a.cnt[0], off_st);
  if (dup) atomicAdd(&a.cnt[3], dup);
  if (pos) atomicAdd(&a.cnt[4], pos);
}

__global__ void __launch_bounds__(256) k_coo_mirror(ImportArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < a.nnz; q += stride) {
    const int64_t i = a.coo_row[q], j = a.col[q];
    bool legal;
    const int slot = coo_slot(a, i, j, &legal);
    if (slot < 4 || !legal) continue;
    const double m = slot == 4 ? a.d1[j] : (slot == 5 ? a.d2[j] : a.d3[j]);      // the mirror is element j of its diagonal
    if (!(a.val[q] == m)) atomicOr(&a.seen[i], 1u << 8);
  }
}

__global__ void __launch_bounds__(256) k_coo_rows(ImportArgs a) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  unsigned long long asym = 0, bad = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    const unsigned sn = a.seen[i];
    const int64_t rem = i % a.nxny;
    const bool has_xm = rem % a.nx > 0, has_ym = rem / a.nx > 0;
    const double m1 = i >= 1 ? a.d1[i - 1] : 0.0;
    const double m2 = i >= a.nx ? a.d2[i - a.nx] : 0.0;
    const double m3 = i >= a.nxny ? a.d3[i - a.nxny] : 0.0;
    bool as = (sn >> 8) & 1u;
    // a mirror that is stored non-zero while row i has no lower entry there (absent == 0)
    if (has_xm && !(sn & (1u << 4)) && m1 != 0.0) as = true;
    if (has_ym && !(sn & (1u << 5)) && m2 != 0.0) as = true;
    if (!(sn & (1u << 6)) && m3 != 0.0) as = true;
    if (as) ++asym;
    const double d = a.d0[i];
    if (!(sn & 1u) || !(d > 0.0) || isinf(d)) ++bad;
    rowsum_minmax(a, i, m1, m2, m3);
  }
  if (asym) atomicAdd(&a.cnt[1], asym);
  if (bad) atomicAdd(&a.cnt[2], bad);
}

// fp32 copy A2 (round-to-nearest-even of the packed values) and 1/D0, as the builder writes them.
__global__ void __launch_bounds__(256) k_import_finish(const double* __restrict__ vals, float* __restrict__ f, int64_t e,
                                                       double* __restrict__ dinv, int64_t n) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < e; i += stride) {
    const double v = vals[i];
    f[i] = __double2float_rn(v);
    if (i < n) dinv[i] = __ddiv_rn(1.0, v);
  }
}

static double key_to_double(unsigned long long k) {
  const unsigned long long b = (k >> 63) ? (k & 0x7fffffffffffffffull) : ~k;
  double v;
  memcpy(&v, &b, sizeof v);
  return v;
}

// Host side of cuth_import_csr.  Synchronises `st` (setup call).  rowsum_layer_H may be nullptr.
int launch_import(const cuth_grid_t* g, const DiaLayout& L, const int64_t* rowptr_D, const int32_t* col_D,
                  const double* val_D, const double* rowsum_layer_H, void* dia_D, cuth_import_report_t* rep,
                  cudaStream_t st, cudaError_t* err, const int32_t* coo_row_D, int64_t nnz) {
  char* base = (char*)dia_D;
  const int nz = (int)L.nz;
  const size_t nlay = 4 * (size_t)nz + 4;
  std::vector<unsigned long long> h(nlay, 0ull);
  for (int z = 0; z < nz; ++z) { h[z] = ~0ull; h[2 * nz + z] = ~0ull; }   // min slots start at the largest key
  unsigned long long hdr[kHeaderBytes / 8] = {0};
  hdr[0] = kMagic; hdr[1] = (unsigned long long)L.nx; hdr[2] = (unsigned long long)L.ny;
  hdr[3] = (unsigned long long)L.nz; hdr[4] = (unsigned long long)L.e; hdr[5] = 0ull;
  for (int k = 0; k < 5; ++k) hdr[6 + k] = (unsigned long long)L.ptr[k];
  for (int k = 0; k < 4; ++k) hdr[11 + k] = (unsigned long long)L.off[k];
  hdr[kHdrImported] = 1ull; hdr[kHdrMixedOk] = 0ull;   // MIXED availability is settled at the end of the import
  cudaError_t e = cudaMemcpyAsync(base, hdr, kHeaderBytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(base + L.o_layers, h.data(), nlay * 8, cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
  unsigned long long* lay = (unsigned long long*)(base + L.o_layers);
  double* v = (double*)(base + L.o_vals);
  float* f = (float*)(base + L.o_vals32);
  ImportArgs a;
  a.n = L.n; a.nx = L.nx; a.ny = L.ny; a.nxny = L.nxny; a.nz = nz;
  a.rowptr = rowptr_D; a.col = col_D; a.val = val_D;
  a.d0 = v + L.ptr[0]; a.d1 = v + L.ptr[1]; a.d2 = v + L.ptr[2]; a.d3 = v + L.ptr[3];
  a.cnt = (unsigned long long*)base + 32;     // header words 32..36
  a.rs_min = lay; a.rs_max = lay + nz; a.d0_min = lay + 2 * nz;
  int64_t blocks = (L.n + 255) / 256;
  if (blocks > 148 * 64) blocks = 148 * 64;
  a.coo_row = coo_row_D; a.nnz = nnz; a.seen = (unsigned int*)(base + L.o_dinv);    // scratch until k_import_finish
  if (coo_row_D) {
    e = cudaMemsetAsync(v, 0, sizeof(double) * (size_t)L.e, st);                    // a missing entry is +0.0
    if (e == cudaSuccess) e = cudaMemsetAsync(a.seen, 0, sizeof(unsigned int) * (size_t)L.n, st);
    if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
    int64_t eb = (nnz + 255) / 256;
    if (eb > 148 * 64) eb = 148 * 64;
    if (eb < 1) eb = 1;
    k_coo_scatter<<<(unsigned)eb, 256, 0, st>>>(a);
    k_coo_mirror<<<(unsigned)eb, 256, 0, st>>>(a);
    k_coo_rows<<<(unsigned)blocks, 256, 0, st>>>(a);
  } else {
    unsigned long long bad_rowptr = 0;
    k_import_check_rowptr<<<(unsigned)blocks, 256, 0, st>>>(rowptr_D, L.n, nnz, a.cnt + 5);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad_rowptr, a.cnt + 5, 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
    if (bad_rowptr) {
      if (rep) { rep->bad_rowptr = (int64_t)bad_rowptr; rep->mixed_ok = 0; }
      return CUTH_ERR_STRUCTURE;
    }
    k_import_upper<<<(unsigned)blocks, 256, 0, st>>>(a);
    k_import_lower<<<(unsigned)blocks, 256, 0, st>>>(a);
  }
  k_import_finish<<<(unsigned)blocks, 256, 0, st>>>(v, f, L.e, (double*)(base + L.o_dinv), L.n);
  BuildArgs b;
  memset(&b, 0, sizeof b);
  b.nx = L.nx; b.ny = L.ny; b.nz = L.nz; b.n = L.n; b.nxny = L.nxny;
  b.d0 = a.d0; b.d1 = a.d1; b.d2 = a.d2; b.d3 = a.d3;
  b.dinv = (double*)(base + L.o_dinv);
  b.f0 = f + L.ptr[0]; b.f1 = f + L.ptr[1]; b.f2 = f + L.ptr[2]; b.f3 = f + L.ptr[3];
  double* slot = (double*)(base + L.o_layers) + 4 * nz;
  k_offdiag_absmax<<<(unsigned)blocks, 256, 0, st>>>(a.d1, L.e - L.n, slot);
  k_h16_scale<<<1, 1, 0, st>>>(slot);
  k_make_h16<<<(unsigned)blocks, 256, 0, st>>>(b, slot, (__half*)(base + L.o_h16), (__half*)(base + L.o_h16 + L.h16_stride),
                                               (__half*)(base + L.o_h16 + 2 * L.h16_stride));
  k_make_f32a<<<(unsigned)blocks, 256, 0, st>>>(b, (float*)(base + L.o_f32a), (float*)(base + L.o_f32a + L.f32a_stride),
                                                (float*)(base + L.o_f32a + 2 * L.f32a_stride), (double*)(base + L.o_f64a),
                                                (double*)(base + L.o_f64a + L.f64a_stride),
                                                (double*)(base + L.o_f64a + 2 * L.f64a_stride), (float*)(base + L.o_dinv32));
  e = cudaGetLastError();
  unsigned long long cnt[5];
  if (e == cudaSuccess) e = cudaMemcpyAsync(cnt, a.cnt, sizeof cnt, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(h.data(), lay, 3 * (size_t)nz * 8, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
  // per-layer row sums s(z) of the MIXED operator (difference form, DESIGN.md R-F3): the caller's, else the
  // midrange of the computed row sums of the layer (clamped at 0); usable only if every row of the layer agrees
  // with it to 1e-9 of the layer's smallest diagonal entry.
  std::vector<double> lay_out(4 * (size_t)nz, 0.0);
  double dev = 0.0;
  bool ok = true;
  for (int z = 0; z < nz; ++z) {
    const double lo = key_to_double(h[z]), hi = key_to_double(h[nz + z]), dmin = key_to_double(h[2 * nz + z]);
    double s = rowsum_layer_H ? rowsum_layer_H[z] : 0.5 * (lo + hi);
    if (!rowsum_layer_H && s < 0.0) s = 0.0;
    const double dz = fmax(fabs(hi - s), fabs(lo - s)) / (dmin > 0.0 ? dmin : 1.0);
    if (!(dz <= 1e-9) || !(s >= 0.0)) ok = false;
    if (!(dz <= dev)) dev = dz;
    lay_out[nz + z] = s;
  }
  const bool structure_ok = cnt[0] == 0 && cnt[1] == 0 && cnt[2] == 0 && cnt[3] == 0;
  if (!ok || !structure_ok)
    for (int z = 0; z < nz; ++z) lay_out[nz + z] = nan("");   // second line of defence: a MIXED solve breaks down loudly
  e = cudaMemcpyAsync(lay, lay_out.data(), lay_out.size() * 8, cudaMemcpyHostToDevice, st);
  const unsigned long long mixed_ok = (ok && structure_ok) ? 1ull : 0ull;    // recorded IN the object (device header)
  if (e == cudaSuccess)
    e = cudaMemcpyAsync((unsigned long long*)base + kHdrMixedOk, &mixed_ok, 8, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
  if (rep) {
    rep->off_stencil = (int64_t)cnt[0]; rep->asymmetric_rows = (int64_t)cnt[1]; rep->bad_diagonal = (int64_t)cnt[2];
    rep->duplicates = (int64_t)cnt[3]; rep->positive_offdiag = (int64_t)cnt[4];
    rep->max_rowsum_dev = dev; rep->mixed_ok = (ok && structure_ok) ? 1 : 0;
  }
  if (!structure_ok) return CUTH_ERR_STRUCTURE;
  if (rowsum_layer_H && !ok) return CUTH_ERR_STRUCTURE;
  return CUTH_OK;
}

}  // namespace cuth
