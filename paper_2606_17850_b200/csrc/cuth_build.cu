// cuth_build.cu -- condensed-DIA ("Quad-Diag") builder kernel: hot-path step a0.
// One thread per cell evaluates eq. (4)/(5) and writes the main and the
// three upper diagonals, the fp32 copy A2, and 1/D0.  Every fp64 operation is an explicit
// round-to-nearest intrinsic (no FMA contraction), in the order stated in DESIGN.md §4, so the
// stored values can be compared bit for bit with an independently assembled matrix.
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
__global__ void __launch_bounds__(256) k_make_f32a(BuildArgs a, float* g1, float* g2, float* g3) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += stride) {
    g1[i] = i + 1 < a.n ? a.f1[i] : 0.f;
    g2[i] = i + a.nx < a.n ? a.f2[i] : 0.f;
    g3[i] = i + a.nxny < a.n ? a.f3[i] : 0.f;
  }
}

// Host side: fills the per-layer arrays, launches the kernel.  Called from cuth_api.cu.
int launch_build(const cuth_grid_t* g, const DiaLayout& L, void* dia_D, cudaStream_t st, cudaError_t* err) {
  char* base = (char*)dia_D;
  const int nz = (int)g->nz;
  const bool transient = g->cvol_H != nullptr && g->dt > 0.0;
  // per-layer arrays inside the matrix object: dz | s | cap | cvol
  double* h = new double[4 * nz + 4];
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
  cudaError_t e = cudaMemcpyAsync(base, hdr, kHeaderBytes, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(base + L.o_layers, h, (4 * nz + 4) * sizeof(double), cudaMemcpyHostToDevice, st);
  delete[] h;   // pageable H2D copies are staged before cudaMemcpyAsync returns
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
                                                (float*)(base + L.o_f32a + 2 * L.f32a_stride));
  e = cudaGetLastError();
  if (e != cudaSuccess) { *err = e; return CUTH_ERR_CUDA; }
  return CUTH_OK;
}

}  // namespace cuth
