// cuth_api.cu -- the C ABI of include/cuth.h: argument checks, CUDA-graph construction, launches.
// The PCG loop is ONE CUDA graph per workspace.  Nothing in it synchronises with the host.
//   small planes (flat traversal):  k_init -> WHILE{ k_pupdate, k_spmv_dot, k_update<x>,
//                                   IF{ k_true_resid, k_restart } } -> k_finalize
//   large planes (fused path):      k_init -> WHILE{ k_fused_pspmv, k_update<no x>,
//                                   IF{ k_flush_x, k_true_resid, k_restart } } -> k_finalize
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <unordered_map>
#include <vector>

#include "cuth_fused.cuh"
#include "cuth_fused_x2.cuh"
#include "cuth_cheb.cuh"
#include "cuth_cheb_pair.cuh"
#include "cuth_cheb_pair_tma.cuh"
#include "cuth_fused_tma.cuh"
#include "cuth_spmv_tma.cuh"
#include "cuth_persistent.cuh"
#include "cuth_fixed32.cuh"
#include "cuth_cluster.cuh"
#include "cuth_cluster_reg.cuh"
#include "cuth_batch.cuh"

namespace cuth {

int launch_build(const cuth_grid_t* g, const DiaLayout& L, void* dia_D, cudaStream_t st, cudaError_t* err);
int launch_import(const cuth_grid_t* g, const DiaLayout& L, const int64_t* rowptr_D, const int32_t* col_D,
                  const double* val_D, const double* rowsum_layer_H, void* dia_D, cuth_import_report_t* rep,
                  cudaStream_t st, cudaError_t* err, const int32_t* coo_row_D = nullptr, int64_t nnz = 0);

static thread_local std::string g_last_err;

static int cuda_fail(cudaError_t e, const char* what) {
  char buf[256];
  snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
  g_last_err = buf;
  cudaGetLastError();
  return CUTH_ERR_CUDA;
}
#define CU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return cuda_fail(e_, #x); } while (0)

static bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

// Kernel variants of one call (cuth_tuning_t, validated): nothing here is process-wide.
struct Tune {
  int traversal = 0;    // 0 auto, 1 flat, 2 z-march
  int loop_mode = 0;    // 0 auto, 1 CUDA graph, 2 persistent cooperative kernel, 3 cluster-resident kernel, 4 its shared-memory form
  int k1_variant = 0;   // 0 auto, 1 one column per thread, 2 two columns, 3 two columns without the TMA-staged K1
  int cheb_pairs = 0;   // 0 auto, 1 never, 2 always (fp32 modes)
  int pair_tma = 0;     // 0 auto (TMA when possible), 1 never
  int pair_rows = 0;    // 0 auto, 8, 16
  int pair_occ = 0;     // 0 auto (4), 2..4
  int lanczos_fp32 = 0; // 1: the paper's fp32 Lanczos on A2
};
static int make_tune(const cuth_tuning_t* t, Tune* T) {
  *T = Tune();
  if (!t) return CUTH_OK;
  if (t->traversal < 0 || t->traversal > 2 || t->loop_mode < 0 || t->loop_mode > 4 || t->k1_variant < 0 ||
      t->k1_variant > 3 || t->cheb_fusion < 0 || t->cheb_fusion > 3 ||
      (t->pair_rows != 0 && t->pair_rows != 8 && t->pair_rows != 16) ||
      (t->pair_occupancy != 0 && (t->pair_occupancy < 2 || t->pair_occupancy > 4)) || t->lanczos_fp32 < 0 ||
      t->lanczos_fp32 > 1 || t->reserved)
    return CUTH_ERR_VALUE;
  T->traversal = t->traversal; T->loop_mode = t->loop_mode; T->k1_variant = t->k1_variant;
  T->cheb_pairs = t->cheb_fusion == 3 ? 2 : t->cheb_fusion;
  T->pair_tma = t->cheb_fusion == 3 ? 1 : 0;
  T->pair_rows = t->pair_rows; T->pair_occ = t->pair_occupancy; T->lanczos_fp32 = t->lanczos_fp32;
  return CUTH_OK;
}

static int check_grid(const cuth_grid_t* g, DiaLayout* L) {
  if (!g) return CUTH_ERR_NULL;
  if (!make_layout(g, L)) return CUTH_ERR_DIMS;
  if (!(g->dx > 0.0) || !(g->dy > 0.0) || !(g->h_top >= 0.0)) return CUTH_ERR_VALUE;
  return CUTH_OK;
}

// Traversal choice: the flat kernel relies on L2 to keep the +-nx*ny neighbours (two planes of six
// arrays, 96 B per plane cell); beyond ~1/3 of the 126 MB L2 that fails and z-marching wins.  On grids whose
// vectors do not fit L2 anyway (> 2^21 rows) the fused two-kernel iteration of the z-marching path (8m + 80 B/row
// against 8m + 104) already pays from 2^17 columns on: measured per Jacobi iteration, flat / z-marching,
// 384x384x128 442 / 355 us, 512x256x128 393 / 329, 448x448x64 312 / 279, but 256x256x256 (2^16 columns: too few
// CTAs) 383 / 413; the Chebyshev path is indifferent there (+-3 %).
static bool use_zmarch(const DiaLayout& L, const Tune& T) {
  const int mode = T.traversal;
  if (mode == 1) return false;
  if (mode == 2) return true;
  return L.nxny >= (1 << 18) || (L.nxny >= (1 << 17) && L.n > (1 << 21));
}

// Two columns per thread halve the number of CTAs: worth it only while the grid still has several waves
// (cfg 5, 512x512 columns: 512 CTAs on 444 slots ran 13 % slower than the one-column kernel's 1024 CTAs).
static bool enough_tiles_x2(const DiaLayout& L, int wx, int wy) {
  return ((L.nx + wx - 1) / wx) * ((L.ny + wy - 1) / wy) >= 2048;
}
static bool fused_x2(const DiaLayout& L, const Tune& T) {
  const int mode = T.k1_variant;
  if (L.nx % 2 != 0 || mode == 1) return false;
  return mode >= 2 || enough_tiles_x2(L, XTX, XTY);
}
static bool zmarch_x2(const DiaLayout& L, const Tune& T) {
  const int mode = T.k1_variant;
  if (L.nx % 2 != 0 || mode == 1) return false;
  return mode >= 2 || enough_tiles_x2(L, 2 * ZTX, ZTY);
}

static int stencil_blocks(const DiaLayout& L, const Tune& T) {
  if (!use_zmarch(L, T)) return -1;
  const int64_t wx = zmarch_x2(L, T) ? 2 * ZTX : ZTX;         // two columns per thread (even nx, enough tiles)
  const int64_t tiles = ((L.nx + wx - 1) / wx) * ((L.ny + ZTY - 1) / ZTY);
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}

static int grid_blocks(int64_t n);

// Threads per CTA of K2 (k_update<false>); see k2_blocks.
#ifndef CUTH_K2_THREADS
#define CUTH_K2_THREADS 512
#endif
constexpr int kK2Threads = CUTH_K2_THREADS;

// fp32 Chebyshev middle step with two x-adjacent columns per thread: large planes with even nx
static bool cheb_x2(const DiaLayout& L, const Tune& T);
static int cheb_x2_blocks(const DiaLayout& L) {
  const int64_t tiles = ((L.nx + 2 * ZTX - 1) / (2 * ZTX)) * ((L.ny + ZTY - 1) / ZTY);
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}

static int cheb_blocks(const DiaLayout& L, const Tune& T) {
  if (!use_zmarch(L, T)) return grid_blocks(L.n);
  const int64_t tiles = ((L.nx + ZTX - 1) / ZTX) * ((L.ny + CUTH_CHEB_NC * ZTY - 1) / (CUTH_CHEB_NC * ZTY));
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}

static bool cheb_x2(const DiaLayout& L, const Tune& T) { return use_zmarch(L, T) && zmarch_x2(L, T); }

static int fused_blocks(const DiaLayout& L, const Tune& T) {
  if (fused_x2(L, T)) {
    const int64_t t2 = ((L.nx + XTX - 1) / XTX) * ((L.ny + XTY - 1) / XTY);
    return (int)(t2 < kMaxBlocks ? t2 : kMaxBlocks);
  }
  const int64_t tiles = ((L.nx + FTX - 1) / FTX) * ((L.ny + FTY - 1) / FTY);
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}

static DiaDev dev_view(const void* dia_D, const DiaLayout& L, const Tune& T) {
  const char* base = (const char*)dia_D;
  const double* v = (const double*)(base + L.o_vals);
  const float* f = (const float*)(base + L.o_vals32);
  const double* lay = (const double*)(base + L.o_layers);
  DiaDev A;
  A.d0 = v + L.ptr[0]; A.d1 = v + L.ptr[1]; A.d2 = v + L.ptr[2]; A.d3 = v + L.ptr[3];
  A.f0 = f + L.ptr[0];
  A.f1 = (const float*)(base + L.o_f32a);
  A.f2 = (const float*)(base + L.o_f32a + L.f32a_stride);
  A.f3 = (const float*)(base + L.o_f32a + 2 * L.f32a_stride);
  A.dinv = (const double*)(base + L.o_dinv);
  A.dinv32 = (const float*)(base + L.o_dinv32);
  A.h1 = (const __half*)(base + L.o_h16);
  A.h2 = (const __half*)(base + L.o_h16 + L.h16_stride);
  A.h3 = (const __half*)(base + L.o_h16 + 2 * L.h16_stride);
  A.h_scale = lay + 4 * L.nz;
  A.s_layer = lay + L.nz;
  A.cap_layer = lay + 2 * L.nz;
  A.hdr = (const unsigned long long*)base;
  A.n = L.n; A.nx = L.nx; A.nxny = L.nxny;
  A.ny = (int32_t)L.ny; A.nz = (int32_t)L.nz;
  A.zmarch = use_zmarch(L, T) ? 1 : 0;
  A.x2 = zmarch_x2(L, T) ? 1 : 0;
  return A;
}

static int grid_blocks(int64_t n) {
  int64_t b = (n + (int64_t)kThreads * kRows - 1) / ((int64_t)kThreads * kRows);
  const int64_t cap = 148 * 8;           // 8 resident CTAs of 256 threads per SM, one wave
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int)b;
}

// Chebyshev kernels by arithmetic / matrix storage: 0 = fp64 on A1, 1 = fp32 on A2, 2 = fp32 on the fp16 copy A3.
static int cheb_code(const cuth_opts_t* o) {
  if (o->precision != CUTH_MIXED) return 0;
  return o->cheb_storage == CUTH_CHEB_A3_FP16 ? 2 : 1;
}
static void* cheb_first_fn(int code) {
  return code == 0 ? (void*)k_cheb_first<double, MatF32> : code == 1 ? (void*)k_cheb_first<float, MatF32>
                                                                     : (void*)k_cheb_first<float, MatF16>;
}
static void* cheb_mid_fn(int code, bool x2) {
  if (code == 0) return (void*)k_cheb_mid<double, MatF32>;
  if (x2) return code == 1 ? (void*)k_cheb_mid_f32x2<MatF32> : (void*)k_cheb_mid_f32x2<MatF16>;
  return code == 1 ? (void*)k_cheb_mid<float, MatF32> : (void*)k_cheb_mid<float, MatF16>;
}
static void* cheb_pair_fn(int code) {
  return code == 2 ? (void*)k_cheb_pair_f32<MatF16> : (void*)k_cheb_pair_f32<MatF32>;
}
static int cheb_pair_blocks(const DiaLayout& L) {
  const int64_t tiles = ((L.nx + QIX - 1) / QIX) * ((L.ny + QIY - 1) / QIY);
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}
static bool cheb_pairs(const DiaLayout& L, int code, const Tune& T) {
  const int mode = T.cheb_pairs;
  // fp32 arithmetic, column pairs: nx even.  Measured faster on every grid (cfg 2 23.5 -> 21.0 ms, cfg 3 0.92 ->
  // 0.63 s, cfg 4 10.8 -> 7.9 s, cfg 5 5.8 -> 4.3 s, cfg 6 41 -> 34 ms), so automatic = always.
  return code != 0 && mode != 1 && (L.nx & 1) == 0;
}
struct ChebOp { int kind; int step, old, cur, w, y; };     // kind 0 = single MID, 1 = fused pair, 2 = LAST, 3 = MID + LAST
// ---- TMA version of the two-pass kernel: tensor maps over (x, y, z) for its six operand streams
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}
static bool cheb_pairs_tma(const DiaLayout& L, int code, const Tune& T) {
  if (!cheb_pairs(L, code, T) || T.pair_tma == 1) return false;
  const int64_t elems16 = code == 2 ? 8 : 4;           // tensor-map strides are multiples of 16 bytes
  return (L.nx % elems16) == 0 && encode_tiled_fn() != nullptr;
}
// box of `rows` rows x (QX + 16 bytes of) columns x 1 plane of an (nx, ny, nz) array of fp32 / fp16 elements; cells outside
// the array read as zero
static bool make_box_map(CUtensorMap* m, const void* base, bool half, const DiaLayout& L, int rows) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint64_t es = half ? 2 : 4;
  const cuuint64_t dims[3] = {(cuuint64_t)L.nx, (cuuint64_t)L.ny, (cuuint64_t)L.nz};
  const cuuint64_t strides[2] = {(cuuint64_t)L.nx * es, (cuuint64_t)L.nxny * es};
  const cuuint32_t box[3] = {(cuuint32_t)(QX + 16 / (int)es), (cuuint32_t)rows, 1u};   // PairBox<E>::W
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  return enc(m, half ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(base),
             dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
             CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
struct PairMaps { CUtensorMap u, v, r, f1, f2, f3; };
static bool make_pair_maps(PairMaps* pm, const DiaLayout& L, const void* dia_D, const Workspace& w, int code,
                           int old, int cur, int ry) {
  const DiaDev A = dev_view(dia_D, L, Tune());
  const void* cd[4] = {w.cd0, w.cd1, w.cd2, w.cd3};
  const bool h = code == 2;
  return make_box_map(&pm->u, cd[cur], false, L, ry + 2) && make_box_map(&pm->v, cd[old], false, L, ry) &&
         make_box_map(&pm->r, w.crc, false, L, ry) &&
         make_box_map(&pm->f1, h ? (const void*)A.h1 : (const void*)A.f1, h, L, ry) &&
         make_box_map(&pm->f2, h ? (const void*)A.h2 : (const void*)A.f2, h, L, ry + 1) &&
         make_box_map(&pm->f3, h ? (const void*)A.h3 : (const void*)A.f3, h, L, ry);
}
static void* cheb_pair_tma_fn(int code, bool last, int ry) {
  if (ry == 16) {
    if (last) return code == 2 ? (void*)k_cheb_pair_tma<MatF16, true, 16> : (void*)k_cheb_pair_tma<MatF32, true, 16>;
    return code == 2 ? (void*)k_cheb_pair_tma<MatF16, false, 16> : (void*)k_cheb_pair_tma<MatF32, false, 16>;
  }
  if (last) return code == 2 ? (void*)k_cheb_pair_tma<MatF16, true, 8> : (void*)k_cheb_pair_tma<MatF32, true, 8>;
  return code == 2 ? (void*)k_cheb_pair_tma<MatF16, false, 8> : (void*)k_cheb_pair_tma<MatF32, false, 8>;
}
// Region height of the TMA kernel: 16 rows (512 threads) recompute a sixth less than 8 rows; taken when the
// plane still gives every SM several regions.  cuth_tuning_t.pair_rows forces it.
static int pair_tma_rows(const DiaLayout& L, const Tune& T) {
  const int forced = T.pair_rows;
  if (forced == 8 || forced == 16) return forced;
  const int64_t tiles16 = ((L.nx + QIX - 1) / QIX) * ((L.ny + 13) / 14);
  return tiles16 >= 4 * 296 ? 16 : 8;
}
static int pair_tma_blocks(const DiaLayout& L, int ry) {
  const int64_t tiles = ((L.nx + QIX - 1) / QIX) * ((L.ny + ry - 3) / (ry - 2));
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}
// Resident CTAs per SM of the TMA two-pass kernel: built for 4 (64 registers, 47 KB of shared memory).  Fewer can
// be forced (by requesting unused dynamic shared memory at launch) to study the partly filled last wave of
// regions -- cfg 3 has 3078 regions = 5.2 waves of 592 but 6.9 waves of 444.  Measured: occupancy wins over wave
// rounding (pair launch at cfg 3: 0.103 ms with 4, 0.109 with 3, 0.133 with 2; cfg 4: 0.73 / 0.83 ms), so
// automatic = 4.
static int pair_tma_occupancy(const Tune& T) {
  const int forced = T.pair_occ;
  return (forced >= 2 && forced <= 4) ? forced : 4;
}
static unsigned pair_tma_dyn_smem(const Tune& T, int code, int ry) {
  size_t need;
  if (ry == 16) need = code == 2 ? sizeof(PairSmem<__half, 16>) : sizeof(PairSmem<float, 16>);
  else need = code == 2 ? sizeof(PairSmem<__half, 8>) : sizeof(PairSmem<float, 8>);
  const int full_occ = ry == 16 ? 2 : 4, occ = pair_tma_occupancy(T) * full_occ / 4;
  if (occ >= 1 && occ < full_occ) {                   // forced lower occupancy: too much for occ + 1 CTAs
    const size_t per_cta = (size_t)(227 * 1024) / (size_t)(occ + 1) + 1024;
    if (per_cta > need) need = per_cta;
  }
  for (int last = 0; last < 2; ++last)
    cudaFuncSetAttribute(cheb_pair_tma_fn(code, last != 0, ry), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need);
  return (unsigned)need;
}

// ---- TMA-staged K1 (cuth_fused_tma.cuh): tensor maps over (x, y, z) for r, p, p2, 1/D0, D0 and the two sets of
// aligned per-diagonal off-diagonals (fp32 A2, fp64 A1)
static bool make_map3d(CUtensorMap* m, const void* base, int elem_bytes, const DiaLayout& L, int box_w, int box_rows) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  const cuuint64_t es = (cuuint64_t)elem_bytes;
  const cuuint64_t dims[3] = {(cuuint64_t)L.nx, (cuuint64_t)L.ny, (cuuint64_t)L.nz};
  const cuuint64_t strides[2] = {(cuuint64_t)L.nx * es, (cuuint64_t)L.nxny * es};
  const cuuint32_t box[3] = {(cuuint32_t)box_w, (cuuint32_t)box_rows, 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  return enc(m, elem_bytes == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
             const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
             CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
static bool make_k1_maps(K1Maps* km, K1Maps* km64, const DiaLayout& L, const void* dia_D, const Workspace& w) {
  const DiaDev A = dev_view(dia_D, L, Tune());
  const char* base = (const char*)dia_D;
  const void* e1 = base + L.o_f64a;
  const void* e2 = base + L.o_f64a + L.f64a_stride;
  const void* e3 = base + L.o_f64a + 2 * L.f64a_stride;
  return make_map3d(&km->z, w.r, 8, L, K1VW, K1VH) && make_map3d(&km->p, w.p, 8, L, K1VW, K1VH) &&
         make_map3d(&km->p2, w.p2, 8, L, K1VW, K1VH) && make_map3d(&km->d, A.dinv32, 4, L, K1VW + 4, K1VH) &&
         make_map3d(&km->m1, A.f1, 4, L, K1Stage<true>::W1, K1Y) && make_map3d(&km->m2, A.f2, 4, L, K1X, K1Y + 1) &&
         make_map3d(&km->m3, A.f3, 4, L, K1X, K1Y) &&
         make_map3d(&km64->d, A.d0, 8, L, K1VW, K1VH) && make_map3d(&km64->m1, e1, 8, L, K1Stage<false>::W1, K1Y) &&
         make_map3d(&km64->m2, e2, 8, L, K1X, K1Y + 1) && make_map3d(&km64->m3, e3, 8, L, K1X, K1Y);
}
static unsigned k1_tma_dyn_smem() {
  const size_t need = sizeof(K1Smem<true>) > sizeof(K1Smem<false>) ? sizeof(K1Smem<true>) : sizeof(K1Smem<false>);
  cudaFuncSetAttribute((const void*)k_fused_pspmv_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need);
  return (unsigned)need;
}
// K1 takes its operands through TMA when it runs two columns per thread (nx even, enough tiles), nx % 4 == 0 (strides of
// the fp32 tensors), z is r (no Chebyshev), the driver can encode tensor maps, and the variant is not forced away.
// Automatic: from one wave of 64 x 8 tiles on (2 CTAs/SM x 148 SMs = 296; the kernel is persistent over tiles and
// keeps its TMA ring running across them, so it does not need the >= 2048 tiles of the LDG two-column kernel).
// Measured per iteration, graph loop, MIXED, TMA K1 / one-column LDG K1: 512x512x16 84.3 / 108.3 us, 768x768x8
// 92.1 / 119.7, 640x640x10 83.0 / 107.5, 384x384x32 91.2 / 112.0, but 256x256x64 (128 tiles) 104.8 / 155.4 with the
// persistent kernel at 101.1 (profiles/r2c_loop_homes.md).
static bool fused_tma(const DiaLayout& L, const Tune& T, bool cheb) {
  if (cheb || T.k1_variant == 1 || T.k1_variant == 3) return false;
  if ((L.nx % 4) != 0 || encode_tiled_fn() == nullptr) return false;
  if (T.k1_variant == 2) return true;
  return ((L.nx + K1X - 1) / K1X) * ((L.ny + K1Y - 1) / K1Y) >= 288;
}
// persistent over tiles: as many CTAs as are resident (2 per SM), never more than tiles
static int fused_tma_blocks(const DiaLayout& L);

// one two-pass launch outside a graph (cuth_cheb_apply, cuth_profile_kernel)
static cudaError_t launch_pair(const DiaLayout& L, const Tune& T, const void* dia_D, const Workspace& w, int code,
                               const ChebOp& op, cudaStream_t st) {
  Ctx* ctxp = w.ctx; Ctl* ctlp = w.ctl; double* part = w.partials;
  int step = op.step, old = op.old, cur = op.cur, wo = op.w, yo = op.y;
  PairMaps pm;
  const int ry = pair_tma_rows(L, T);
  if (cheb_pairs_tma(L, code, T) && make_pair_maps(&pm, L, dia_D, w, code, old, cur, ry)) {
    void* a[] = {&ctxp, &ctlp, &part, &step, &wo, &yo, &pm.u, &pm.v, &pm.r, &pm.f1, &pm.f2, &pm.f3};
    return cudaLaunchKernel(cheb_pair_tma_fn(code, op.kind == 3, ry), dim3(pair_tma_blocks(L, ry)), dim3(32 * ry), a,
                            pair_tma_dyn_smem(T, code, ry), st);
  }
  if (op.kind == 3) return cudaErrorInvalidValue;      // the fused MID + LAST launch exists only as a TMA kernel
  void* a[] = {&ctxp, &step, &old, &cur, &wo, &yo};
  return cudaLaunchKernel(cheb_pair_fn(code), dim3(cheb_pair_blocks(L)), dim3(kThreads), a, 0, st);
}

static void* cheb_last_fn(int code) {
  return code == 0 ? (void*)k_cheb_last<double, MatF32> : code == 1 ? (void*)k_cheb_last<float, MatF32>
                                                                    : (void*)k_cheb_last<float, MatF16>;
}

// The passes of one Chebyshev apply after the first one: MID passes i = 1 .. k-3 (single, or fused in pairs),
// then LAST (i = k-2).  State = which buffers hold Z_i (old) and Z_{i+1} (cur); k_cheb_first leaves old = 1, cur = 0.
// kind 3 (only with the TMA kernel, fuse_last): the odd MID pass left over by the pairing and LAST in one launch.
static std::vector<ChebOp> cheb_schedule(int k, bool pairs, bool fuse_last) {
  std::vector<ChebOp> ops;
  int old = 1, cur = 0, i = 1;
  while (i <= k - 3) {
    if (pairs && fuse_last && i == k - 3) {
      ops.push_back({3, i, old, cur, -1, -1});
      return ops;
    }
    if (pairs && i + 1 <= k - 3) {
      int fr[2], nf = 0;
      for (int b = 0; b < 4; ++b) if (b != old && b != cur) fr[nf++] = b;
      ops.push_back({1, i, old, cur, fr[0], fr[1]});
      old = fr[0]; cur = fr[1]; i += 2;
    } else {
      ops.push_back({0, i, old, cur, -1, -1});
      const int t = old; old = cur; cur = t; i += 1;
    }
  }
  ops.push_back({2, k - 2, old, cur, -1, -1});
  return ops;
}

// ------------------------------------------------------------------------------------------
// Everything that determines the SHAPE of the graph of a solve (kernels, grids, baked tensor maps, workspace
// layout): the key of the graph cache.  Per-call pointers and options travel in Ctx, not in the graph.
struct Plan {
  int64_t n = 0;
  int sblocks = 0;       // grid of the kernels that apply A (z-marching tiles, or the flat grid)
  int fblocks = 0;       // > 0: fused path (K1 + K2); grid of K1
  int k1x2 = 0;          // K1 with two columns per thread
  int chebkey = 0;       // degree * 4 + arithmetic code, 0 = no Chebyshev preconditioner
  int cblocks = 0, x2blocks = 0, pblocks = 0;    // Chebyshev single-pass / two-column / two-pass grids
  int with_b = 0;        // transient matrix: b lives in the workspace, the Chebyshev buffers sit N doubles later
  int pair_tma = 0;      // the two-pass Chebyshev nodes are the TMA kernel
  int k1tma = 0;         // K1 is the TMA-staged kernel
  int k1dual = 0;        // ... in the early stage only; in the late stage K1 is the two-column LDG kernel (fblocks2 CTAs)
  int fblocks2 = 0;
  int unroll = 1;        // K1 + K2 pairs per pass of the WHILE body (fused path without Chebyshev)
  int k2blocks = 0;      // grid of K2 (one resident wave)
  const void* dia = nullptr;   // matrix the tensor maps of the TMA nodes were made for (else nullptr)
  int64_t tnx = 0, tny = 0;    // ... and its plane dimensions
  int tocc = 0;                // ... occupancy * 100 + region rows of the TMA two-pass nodes
  int device = -1;
  bool operator==(const Plan& o) const {
    return n == o.n && sblocks == o.sblocks && fblocks == o.fblocks && k1x2 == o.k1x2 && chebkey == o.chebkey &&
           cblocks == o.cblocks && x2blocks == o.x2blocks && pblocks == o.pblocks && with_b == o.with_b &&
           pair_tma == o.pair_tma && k1tma == o.k1tma && k1dual == o.k1dual && fblocks2 == o.fblocks2 && unroll == o.unroll && k2blocks == o.k2blocks && dia == o.dia && tnx == o.tnx && tny == o.tny && tocc == o.tocc && device == o.device;
  }
};
struct GraphEntry {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  Plan plan;
};
static std::mutex g_mu;
static std::unordered_map<const void*, GraphEntry> g_graphs;
static std::unordered_map<const void*, const void*> g_last_dia;   // workspace -> matrix of its last solve (profile hook)

static cudaError_t add_kernel(cudaGraph_t g, cudaGraphNode_t* node, const cudaGraphNode_t* deps, size_t ndeps,
                              void* func, int blocks, void** args, unsigned dyn_smem = 0, int threads = kThreads) {
  cudaKernelNodeParams kp;
  memset(&kp, 0, sizeof kp);
  kp.func = func;
  kp.gridDim = dim3((unsigned)blocks);
  kp.blockDim = dim3((unsigned)threads);
  kp.sharedMemBytes = dyn_smem;
  kp.kernelParams = args;
  return cudaGraphAddKernelNode(node, g, deps, ndeps, &kp);
}

static int build_graph(const Workspace& w, const Plan& P, const DiaLayout& L, const Tune& T, GraphEntry* out) {
  const int blocks = grid_blocks(P.n);
  const int sblocks = P.sblocks;
  cudaGraph_t g;
  CU(cudaGraphCreate(&g, 0));
  cudaGraphConditionalHandle h_while, h_if;
  CU(cudaGraphConditionalHandleCreate(&h_while, g, 0, cudaGraphCondAssignDefault));
  CU(cudaGraphConditionalHandleCreate(&h_if, g, 0, cudaGraphCondAssignDefault));
  Ctx* ctx = w.ctx; Ctl* ctl = w.ctl; double* partials = w.partials;

  cudaGraphNode_t n_init, n_while, n_fin;
  { void* a[] = {&ctx, &ctl, &partials, &h_while};
    CU(add_kernel(g, &n_init, nullptr, 0, (void*)k_init, sblocks, a)); }
  cudaGraphNodeParams wp = {};
  wp.type = cudaGraphNodeTypeConditional;
  wp.conditional.handle = h_while;
  wp.conditional.type = cudaGraphCondTypeWhile;
  wp.conditional.size = 1;
  CU(cudaGraphAddNode(&n_while, g, &n_init, 1, &wp));
  cudaGraph_t body = wp.conditional.phGraph_out[0];
  { void* a[] = {&ctx, &ctl};
    CU(add_kernel(g, &n_fin, &n_while, 1, (void*)k_finalize, blocks, a)); }

  cudaGraphNode_t n_p, n_s, n_u, n_if;
  // Chebyshev: the body starts with the preconditioner z = q(A) r: k-1 stencil kernels, no reduction
  // until the last one, which also forms rho = r.z and beta (Alg. 1 lines 10-11).
  cudaGraphNode_t n_c = nullptr;
  const int kdeg = P.chebkey >> 2;
  if (kdeg > 0) {
    const int code = P.chebkey & 3;
    const bool f32 = code != 0;
    { void* a[] = {&ctx};
      CU(add_kernel(body, &n_c, nullptr, 0, cheb_first_fn(code), P.cblocks, a)); }
    for (const ChebOp& op : cheb_schedule(kdeg, P.pblocks > 0, P.pair_tma != 0)) {
      cudaGraphNode_t prev = n_c;
      int step = op.step, old = op.old, cur = op.cur, wo = op.w, yo = op.y;
      PairMaps pm;
      if ((op.kind == 1 || op.kind == 3) && P.pair_tma) {
        const int ry = pair_tma_rows(L, T);
        if (!make_pair_maps(&pm, L, P.dia, w, code, old, cur, ry)) return CUTH_ERR_CUDA;
        void* a[] = {&ctx, &ctl, &partials, &step, &wo, &yo, &pm.u, &pm.v, &pm.r, &pm.f1, &pm.f2, &pm.f3};   // copied into the node
        CU(add_kernel(body, &n_c, &prev, 1, cheb_pair_tma_fn(code, op.kind == 3, ry), pair_tma_blocks(L, ry), a,
                      pair_tma_dyn_smem(T, code, ry), 32 * ry));
      } else if (op.kind == 1) {
        void* a[] = {&ctx, &step, &old, &cur, &wo, &yo};
        CU(add_kernel(body, &n_c, &prev, 1, cheb_pair_fn(code), P.pblocks, a));
      } else if (op.kind == 0) {
        void* a[] = {&ctx, &step, &old, &cur};
        if (f32 && P.x2blocks > 0)
          CU(add_kernel(body, &n_c, &prev, 1, cheb_mid_fn(code, true), P.x2blocks, a));
        else
          CU(add_kernel(body, &n_c, &prev, 1, cheb_mid_fn(code, false), P.cblocks, a));
      } else {
        void* a[] = {&ctx, &ctl, &partials, &step, &old, &cur};
        CU(add_kernel(body, &n_c, &prev, 1, cheb_last_fn(code), P.cblocks, a));
      }
    }
  }
  const cudaGraphNode_t* dep0 = n_c ? &n_c : nullptr;
  const size_t ndep0 = n_c ? 1 : 0;
  if (P.fblocks > 0) {
    // A pass of the WHILE node costs ~9 us of scheduling, so the body holds P.unroll iterations; once
    // K2's epilogue decides that the loop must stop or that the true-residual branch must run (ctl->halt), the
    // remaining K1 / K2 launches of the pass return at once and the IF node at the end of the body takes over.
    K1Maps km, km64;
    if (P.k1tma && !make_k1_maps(&km, &km64, L, P.dia, w)) return CUTH_ERR_CUDA;
    const unsigned k1_smem = P.k1tma ? k1_tma_dyn_smem() : 0u;
    for (int u = 0; u < P.unroll; ++u) {
      const cudaGraphNode_t* dep = u == 0 ? dep0 : &n_u;
      const size_t ndep = u == 0 ? ndep0 : 1;
      if (P.k1tma) {
        void* a[] = {&ctx, &ctl, &partials, &km.z, &km.p, &km.p2, &km.d, &km64.d, &km.m1, &km.m2, &km.m3,
                     &km64.m1, &km64.m2, &km64.m3};                    // the maps are copied into the node
        CU(add_kernel(body, &n_s, dep, ndep, (void*)k_fused_pspmv_tma, P.fblocks, a, k1_smem));
        if (P.k1dual) {        // thin stacks: the late stage's K1 (Ctx.k1_split makes each return in the other's stage)
          cudaGraphNode_t n_e = n_s;
          void* a2[] = {&ctx, &ctl, &partials};
          CU(add_kernel(body, &n_s, &n_e, 1, (void*)k_fused_pspmv_x2, P.fblocks2, a2));
        }
      } else {
        void* a[] = {&ctx, &ctl, &partials};
        CU(add_kernel(body, &n_s, dep, ndep, P.k1x2 ? (void*)k_fused_pspmv_x2 : (void*)k_fused_pspmv, P.fblocks, a));
      }
      void* a2[] = {&ctx, &ctl, &partials, &h_while, &h_if};
      CU(add_kernel(body, &n_u, &n_s, 1, (void*)k_update<false>, P.k2blocks, a2, 0, kK2Threads));
    }
  } else {
    { void* a[] = {&ctx, &ctl};
      CU(add_kernel(body, &n_p, dep0, ndep0, (void*)k_pupdate, blocks, a)); }
    { void* a[] = {&ctx, &ctl, &partials};
      CU(add_kernel(body, &n_s, &n_p, 1, (void*)k_spmv_dot, sblocks, a)); }
    { void* a[] = {&ctx, &ctl, &partials, &h_while, &h_if};
      CU(add_kernel(body, &n_u, &n_s, 1, (void*)k_update<true>, blocks, a)); }
  }
  cudaGraphNodeParams ip = {};
  ip.type = cudaGraphNodeTypeConditional;
  ip.conditional.handle = h_if;
  ip.conditional.type = cudaGraphCondTypeIf;
  ip.conditional.size = 1;
  CU(cudaGraphAddNode(&n_if, body, &n_u, 1, &ip));
  cudaGraph_t ifb = ip.conditional.phGraph_out[0];
  cudaGraphNode_t n_f, n_t, n_r;
  if (P.fblocks > 0) {
    void* a[] = {&ctx, &ctl};
    CU(add_kernel(ifb, &n_f, nullptr, 0, (void*)k_flush_x, blocks, a));
  }
  { void* a[] = {&ctx, &ctl, &partials, &h_while};
    CU(add_kernel(ifb, &n_t, P.fblocks > 0 ? &n_f : nullptr, P.fblocks > 0 ? 1 : 0, (void*)k_true_resid, sblocks, a)); }
  { void* a[] = {&ctx, &ctl, &partials};
    CU(add_kernel(ifb, &n_r, &n_t, 1, (void*)k_restart, sblocks, a)); }      // applies A1 itself: the stencil grid

  cudaGraphExec_t ex;
  CU(cudaGraphInstantiate(&ex, g, 0));
  out->graph = g; out->exec = ex; out->plan = P;
  return CUTH_OK;
}

static int get_graph(const Workspace& w, void* work_D, const Plan& P, const DiaLayout& L, const Tune& T,
                     cudaGraphExec_t* ex) {
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_graphs.find(work_D);
  if (it != g_graphs.end() && !(it->second.plan == P)) {
    cudaGraphExecDestroy(it->second.exec);
    cudaGraphDestroy(it->second.graph);
    g_graphs.erase(it);
    it = g_graphs.end();
  }
  if (it == g_graphs.end()) {
    GraphEntry e;
    int rc = build_graph(w, P, L, T, &e);
    if (rc != CUTH_OK) return rc;
    it = g_graphs.emplace(work_D, e).first;
  }
  *ex = it->second.exec;
  return CUTH_OK;
}

static int check_opts(const cuth_opts_t* o) {
  if (!o) return CUTH_ERR_NULL;
  if (!(o->rtol > 0.0) || o->max_iters <= 0) return CUTH_ERR_VALUE;
  if (o->precision != CUTH_FP64 && o->precision != CUTH_MIXED && o->precision != CUTH_MIXED_STD32 &&
      o->precision != CUTH_FIXED32)
    return CUTH_ERR_VALUE;
  if ((o->precision == CUTH_MIXED_STD32 || o->precision == CUTH_FIXED32) && o->preconditioner == CUTH_PRECOND_CHEBYSHEV)
    return CUTH_ERR_VALUE;                               // ablations: Alg. 1 with M = D0 or I
  Tune T;
  if (make_tune(&o->tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  if (o->preconditioner != CUTH_PRECOND_NONE && o->preconditioner != CUTH_PRECOND_JACOBI &&
      o->preconditioner != CUTH_PRECOND_CHEBYSHEV)
    return CUTH_ERR_VALUE;
  if (o->preconditioner == CUTH_PRECOND_CHEBYSHEV &&
      (o->cheb_degree < 3 || o->cheb_degree > kMaxChebDegree || !(o->cheb_lmin > 0.0) || !(o->cheb_lmax > o->cheb_lmin) ||
       (o->cheb_storage != CUTH_CHEB_DEFAULT && o->cheb_storage != CUTH_CHEB_A3_FP16)))
    return CUTH_ERR_VALUE;
  return CUTH_OK;
}

// Alg. 3 lines 2-3, 9-10 in fp64 on the host: theta, delta, sigma_1, rho_i and the two
// coefficients of line 10 for every step; buffers of the preconditioner.
static void fill_cheb(Ctx* c, const cuth_opts_t* opts, const Workspace& w) {
  const int k = opts->cheb_degree;
  const double theta = 0.5 * (opts->cheb_lmax + opts->cheb_lmin), delta = 0.5 * (opts->cheb_lmax - opts->cheb_lmin);
  const double sigma1 = theta / delta;
  double rho = 1.0 / sigma1;
  for (int i = 0; i < k; ++i) {
    const double rho_next = 1.0 / (2.0 * sigma1 - rho);
    c->cheb_c1[i] = rho_next * rho;
    c->cheb_c2[i] = 2.0 * rho_next / delta;
    rho = rho_next;
  }
  c->cheb = k;
  c->cheb_inv_theta = 1.0 / theta;
  c->cz = w.cz; c->cd[0] = w.cd0; c->cd[1] = w.cd1; c->cd[2] = w.cd2; c->cd[3] = w.cd3; c->crc = w.crc;
  c->jacobi = 0;
  c->precision = opts->precision;
}

// Grid of the persistent kernel: every CTA must be co-resident (cooperative launch).  The grid-wide barrier, not
// the row work, sets the pace on small grids, and its cost is not monotonic in the CTA count: measured per
// iteration at 8 k / 33 k / 66 k / 262 k / 1 M rows with 256-thread CTAs (B200, round 1) -- 32 CTAs
// 11.5 / 16.0 / 22.9 / 51 / 187 us, 96 CTAs 12.4 / 13.9 / 16.0 / 27.7 / 72, 128 CTAs 7.1 / 7.3 / 8.1 / 13.9 / 47, 148 CTAs
// 8.0 / 8.0 / 8.8 / 14.2 / 46, 256 CTAs 9.2 / 8.4 / 8.4 / 12.4 / 33, 592 CTAs 13.4 / 14.1 / 13.7 / 16.7 / 29.8.  Round 2c keeps
// the 128 CTAs and grows the CTAs instead of their number: persistent_config below.
// Co-resident CTAs of a cooperative kernel, per device (derived data, filled on first use under the mutex).
static std::mutex g_dev_mu;
static std::unordered_map<long long, int> g_coresident;      // (device << 8 | kernel slot) -> CTAs
static int coresident_blocks(int slot, const void* fn, int max_per_sm, int cap, size_t dyn_smem = 0, int threads = kThreads) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  std::lock_guard<std::mutex> lk(g_dev_mu);
  const long long key = ((long long)dev << 8) | slot;
  auto it = g_coresident.find(key);
  if (it != g_coresident.end()) return it->second;
  int sms = 0, coop = 0, occ = 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, dyn_smem);
  if (occ > max_per_sm) occ = max_per_sm;
  int v = (coop || slot == 2 || slot >= 4) ? sms * occ : 0;   // slots 2, 4, 5, 6 (TMA K1, K2, TMA SpMV) are ordinary launches
  if (v > cap) v = cap;
  g_coresident[key] = v;
  return v;
}
static int fused_tma_blocks(const DiaLayout& L) {
  const int64_t tiles = ((L.nx + K1X - 1) / K1X) * ((L.ny + K1Y - 1) / K1Y);
  const int resident = coresident_blocks(2, (const void*)k_fused_pspmv_tma, 2, kMaxBlocks, k1_tma_dyn_smem());
  return (int)(tiles < resident ? tiles : (resident > 0 ? resident : 1));
}
// Grid of K2 (k_update<false>, a pure stream): exactly ONE wave of resident CTAs striding over the rows.  Measured at cfg 3
// (B200): 1184 CTAs = two waves 0.0905 ms (late stage) / 0.0849 (early), 592 CTAs = one wave 0.0861 / 0.0809; four instead of
// two row pairs per trip were slower in every combination.  Round 2c: the same wave as 296 CTAs of 512 threads -- half the
// tickets and partials for the last CTA to collect: cfg 3 MIXED 1.3450 / 1.3467 -> 1.3445 s, FP64 1.3728 -> 1.3696 s, cfg 5
// (40 steps) 2.302 -> 2.278 s (1024 threads: 1.3429 / 1.3682 / 2.287).
static int k2_blocks(int64_t n) {
  const int resident = coresident_blocks(4, (const void*)k_update<false>, 2048 / kK2Threads, kMaxBlocks, 0, kK2Threads);
  const int want = (int)((n + (int64_t)kK2Threads * kRows - 1) / ((int64_t)kK2Threads * kRows));
  return resident > 0 && resident < want ? resident : (want > 0 ? want : 1);
}
// Launch configuration of the persistent kernel (and of the fixed-FP32 ablation kernel, which shares its row loops).
// What a grid-wide barrier costs grows with the CTAs that take part in it, so the kernel runs FEW, LARGE CTAs: always 128
// CTAs (a power of two: 148 is slower everywhere), of 256 threads up to 64 k rows, 512 up to 128 k, 1024 beyond (round 2b
// ran 128 / 256 / 592 CTAs of 256 threads up to 64 k / 512 k rows / beyond).  Measured on B200, us per iteration, MIXED,
// 128 CTAs of 256 / 512 / 1024 threads: 8 k rows 6.9 / 7.2 / 8.5; 37 k 7.9 / 8.3 / 9.3; 65 k 8.4 / 8.3 / 9.8; 131 k 10.5 /
// 9.4 / 10.0; 262 k 14.6 / 12.1 / 11.5; cfg 6 (655 k) 25.1 / 17.6 / 16.6; and 1024-thread CTAs x 32 / 64 / 96 / 128 / 148:
// 262 k 21.1 / 17.0 / 15.8 / 11.0 / 12.1; cfg 6 40.2 / 25.4 / 22.3 / 16.3 / 17.1; cfg 2 (1 M) 58.6 / 36.1 / 29.9 / 21.8 /
// 22.1 -- against 12.5 (262 k), 20.3 (cfg 6) and 25.2 (cfg 2) with round 2b's configuration.
struct PersistConfig { int blocks, threads; };
static PersistConfig persistent_config(int64_t n) {
#ifdef CUTH_PERSIST_THREADS
  const int threads = CUTH_PERSIST_THREADS;
#else
  const int threads = n <= (1 << 16) ? 256 : (n <= (1 << 17) ? 512 : kPersistMaxThreads);
#endif
#ifdef CUTH_PERSIST_CTAS
  const int want = CUTH_PERSIST_CTAS;
#else
  const int want = n > 3 * (1 << 19) ? kPersistMaxBlocks : 128;      // beyond 1.5 M rows: every SM (2 M rows: 45.6 vs 48.4 us)
#endif
  const int all = coresident_blocks(0, (const void*)k_pcg_persistent, 1, kPersistMaxBlocks, 0, kPersistMaxThreads);
  return {want < all ? want : all, threads};
}
static int persistent_blocks(int64_t n) { return persistent_config(n).blocks; }

// The cluster-resident kernels (cuth_cluster_reg.cuh, cuth_cluster.cuh): every row lives in the registers / the shared memory
// of one 8- or 16-CTA cluster.  Measured on B200 (profiles/r2e_cluster.md), per iteration, cluster / persistent kernel /
// graph: cfg 1 (8 192 rows) 2.2 / 6.9 / 18.8 us, 2 048 rows 2.1 / 6.4 / 19.4, 12 800 rows 2.7 / 7.2 / 19.2.
static bool use_cluster(const DiaLayout& L, const cuth_opts_t* opts, const Tune& T) {
  if (T.loop_mode == 1 || T.loop_mode == 2 || T.traversal == 2) return false;
  if (opts->preconditioner == CUTH_PRECOND_CHEBYSHEV) return false;
  if (opts->precision != CUTH_FP64 && opts->precision != CUTH_MIXED) return false;
  return cluster_fits(L.nx, L.ny, L.nz, kClusterMaxCtas);
}

// One cluster per solve (nsolves > 1: cuth_pcg_solve_batch, contexts and control blocks as arrays).
// Up to 1024 rows per CTA the rows live in registers (cuth_cluster_reg.cuh); beyond, or with loop_mode = 4, in shared
// memory (cuth_cluster.cuh).  The candidates are tried in the measured order of speed until one launches (a 16-CTA
// cluster is a non-portable size and may be refused).  Measured at cfg 1 (8 192 rows, FP64 / MIXED, us per iteration):
// 16 CTAs x 256 threads 2.17 / 2.32, 16 x 512 (one row per thread) 2.46 / 2.64, 8 x 512 2.59 / 2.78, shared-memory form
// 8 x 1024 3.91 / 4.12 -- FP64 adds, 64-bit shuffles and distributed-shared-memory bytes per SM are the narrow resources,
// so spreading the rows over 16 SMs wins although the all-reduce has twice the partners.  A batch is a different matter:
// a 16-CTA cluster takes a whole GPC where two 8-CTA ones share it, so the form whose (waves of co-resident clusters) x
// (relative time of one solve: 1 for 16 x 256, 1.2 for 8 x 512) is smaller goes first.
struct ClusterForm { int nc, threads; const void* fn; };     // threads = 1024: the shared-memory form
static bool cluster_form_config(const ClusterForm& f, const DiaLayout& L, int nsolves, cudaStream_t st, cudaLaunchConfig_t* cfg,
                                cudaLaunchAttribute* at, int* rows) {
  const bool reg = f.threads != kClusterThreads;
  *rows = (int)cluster_rows_per_cta(L.nx, L.ny, L.nz, f.nc);
  const size_t smem = reg ? cluster_reg_smem_bytes(*rows) : cluster_smem_bytes(*rows);
  if (cudaFuncSetAttribute(f.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
      (f.nc > 8 && cudaFuncSetAttribute(f.fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess)) {
    cudaGetLastError();
    return false;
  }
  memset(cfg, 0, sizeof *cfg);
  cfg->gridDim = dim3((unsigned)(f.nc * nsolves)); cfg->blockDim = dim3((unsigned)f.threads);
  cfg->dynamicSmemBytes = smem; cfg->stream = st;
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = f.nc; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg->attrs = at; cfg->numAttrs = 1;
  return true;
}
// Clusters of this form that can be resident at once on the current device (0: unknown).
static int cluster_form_resident(const ClusterForm& f, const DiaLayout& L) {
  cudaLaunchConfig_t cfg; cudaLaunchAttribute at[1]; int rows = 0, nclu = 0, dev = 0;
  if (!cluster_form_config(f, L, 1, nullptr, &cfg, at, &rows) || cudaGetDevice(&dev) != cudaSuccess) return 0;
  // derived data, cached per (device, form, shared-memory size) like the co-resident CTA counts
  const long long key = ((long long)dev << 40) | ((long long)f.nc << 32) | ((long long)f.threads << 20) | (long long)(rows & 0xfffff);
  static std::unordered_map<long long, int> cache;
  std::lock_guard<std::mutex> lk(g_dev_mu);
  auto it = cache.find(key);
  if (it != cache.end()) return it->second;
  if (cudaOccupancyMaxActiveClusters(&nclu, f.fn, &cfg) != cudaSuccess) { cudaGetLastError(); nclu = 0; }
  cache[key] = nclu;
  return nclu;
}
static cudaError_t launch_cluster(const DiaLayout& L, const Ctx* ctxp, Ctl* ctlp, int nsolves, cudaStream_t st,
                                  bool allow_reg) {
  const ClusterForm r8 = {8, 512, (const void*)k_pcg_cluster_reg<8, 512>}, r16h = {16, 256, (const void*)k_pcg_cluster_reg<16, 256>},
                    r16 = {16, 512, (const void*)k_pcg_cluster_reg<16, 512>}, s8 = {8, kClusterThreads, (const void*)k_pcg_cluster<8>},
                    s16 = {16, kClusterThreads, (const void*)k_pcg_cluster<16>};
  const ClusterForm one[] = {r16h, r8, r16, s8, s16}, many[] = {r8, r16h, r16, s8, s16};
  bool eight_first = false;
  if (nsolves > 1 && allow_reg && cluster_reg_fits(L.nx, L.ny, L.nz, 16, 256) && cluster_reg_fits(L.nx, L.ny, L.nz, 8, 512)) {
    const int c16 = cluster_form_resident(r16h, L), c8 = cluster_form_resident(r8, L);
    if (c16 > 0 && c8 > 0) eight_first = 1.2 * ((nsolves + c8 - 1) / c8) < 1.0 * ((nsolves + c16 - 1) / c16);
    else eight_first = nsolves > 8;
  }
  const ClusterForm (&forms)[5] = eight_first ? many : one;
  cudaError_t e = cudaErrorInvalidValue;
  for (const ClusterForm& f : forms) {
    if (e == cudaSuccess) break;
    const bool reg = f.threads != kClusterThreads;
    if (reg ? !(allow_reg && cluster_reg_fits(L.nx, L.ny, L.nz, f.nc, f.threads)) : !cluster_fits(L.nx, L.ny, L.nz, f.nc)) continue;
    cudaLaunchConfig_t cfg; cudaLaunchAttribute at[1]; int rows = 0;
    if (!cluster_form_config(f, L, nsolves, st, &cfg, at, &rows)) continue;
    void* args[] = {(void*)&ctxp, (void*)&ctlp, (void*)&rows};
    e = cudaLaunchKernelExC(&cfg, f.fn, args);
    if (e != cudaSuccess) cudaGetLastError();
  }
  return e;
}

static bool use_persistent(const DiaLayout& L, bool cheb, const Tune& T) {
  const int mode = T.loop_mode, trav = T.traversal;
  if (cheb || mode == 1 || mode >= 3 || trav == 2) return false;
  if (persistent_blocks(L.n) <= 0) return false;
  if (mode == 2) return !use_zmarch(L, T);        // forced: wherever the flat traversal applies
  // Measured on B200: per iteration, persistent kernel / graph with conditional nodes:
  // 7.0 / 18.7 us at cfg 1 (8 k rows), 19.3 / 30.4 us at cfg 6 (655 k), 23.2 / 34.7 us at cfg 2 (1 M); and on wide
  // planes, against the z-marching graph: 512x512x4 23.2 / 36.1, 512x512x8 47.7 / 60.3, 1024x1024x2 47.0 / 66.1,
  // 512x512x16 (4 M rows, cfg 5) 101.0 / 99.5 in FP64 but 103.9 / 112.6 in MIXED with T = 5 (the true-residual branch
  // is three more kernels and an IF node in the graph, one more phase in the kernel).
  // Round 2, graph with the TMA-staged K1 and four iterations per WHILE pass / persistent kernel: 512x512x8 (2 M rows)
  // 48.2 / 47.9 us (MIXED), 1024x1024x2 53.2 / 47.0, but from 4 M rows on 512x512x16 (cfg 5) 84.3 / 101.8, 1024x512x8
  // 86.3 / 101.2, 640x640x10 83.0 / 99.5, 768x768x8 92.1 / 113.7 (profiles/r2c_loop_homes.md).
  // Auto: the persistent kernel (its row access is flat whatever the plane shape) up to 2^21 rows, and up to 2^22
  // rows where the TMA-staged K1 is not available; the graph everywhere else.
  if (L.n > (1 << 22)) return false;
  if (L.n <= (1 << 21)) return true;
  return !(use_zmarch(L, T) && fused_tma(L, T, false));
}

constexpr int kGraphUnroll = 8;   // iterations per pass of the WHILE body on the fused path

// Thin stacks (nz < 12: nz + 1 steps for nz planes) with the fp64 operator: the two-column LDG K1 beats the TMA-staged one
// (cfg 4, nz = 8: 1.66 vs 1.82 ms; FP64 solve 23.45 vs 24.00 s), while with the fp32-stored operator the TMA-staged one wins
// (1.57 ms).  Automatic choice only (k1_variant 0), where both kernels serve the grid:
// 0 = nothing to do, 1 = FP64 solve: LDG K1 throughout, 2 = MIXED solve: TMA K1 in the early stage, LDG K1 in the late one.
static int k1_thin_stack(const DiaLayout& L, const Tune& T, const cuth_opts_t* opts) {
  if (T.k1_variant != 0 || L.nz >= 12 || opts->preconditioner == CUTH_PRECOND_CHEBYSHEV || !fused_x2(L, T)) return 0;
  if (!fused_tma(L, T, false)) return 0;
  return opts->precision == CUTH_FP64 ? 1 : (opts->precision == CUTH_MIXED ? 2 : 0);
}

// The graph of a solve with these options on this grid.
static Plan make_plan(const DiaLayout& L, const Tune& T, const cuth_opts_t* opts, bool with_b, const void* dia_D) {
  Plan P;
  const bool cheb = opts->preconditioner == CUTH_PRECOND_CHEBYSHEV;
  const int code = cheb_code(opts);
  const bool zm = use_zmarch(L, T);
  P.n = L.n;
  const int sb = stencil_blocks(L, T);
  P.sblocks = sb > 0 ? sb : grid_blocks(L.n);
  P.fblocks = zm ? fused_blocks(L, T) : 0;
  P.k1x2 = (zm && fused_x2(L, T)) ? 1 : 0;
  if (zm && fused_tma(L, T, cheb)) {
    P.k1tma = 1; P.fblocks = fused_tma_blocks(L);
    P.dia = dia_D; P.tnx = L.nx; P.tny = L.ny;
    const int split = k1_thin_stack(L, T, opts);
    if (split == 1) { P.k1tma = 0; P.fblocks = fused_blocks(L, T); P.dia = nullptr; P.tnx = P.tny = 0; }
    else if (split == 2) { P.k1dual = 1; P.fblocks2 = fused_blocks(L, T); }
  }
  P.chebkey = cheb ? opts->cheb_degree * 4 + code : 0;
  P.cblocks = cheb_blocks(L, T);
  P.x2blocks = cheb_x2(L, T) ? cheb_x2_blocks(L) : 0;
  P.pblocks = (cheb && cheb_pairs(L, code, T)) ? cheb_pair_blocks(L) : 0;
  P.with_b = with_b ? 1 : 0;
  P.unroll = (P.fblocks > 0 && !cheb) ? kGraphUnroll : 1;
  if (P.unroll > 1 && (opts->precision == CUTH_MIXED || opts->precision == CUTH_MIXED_STD32)) {
    // Early stage: every `period` iterations the pass ends in the true-residual branch.  A body whose length divides
    // the period has no halted (no-op) launches in front of that branch: T = 20 (steady) -> 10, T = 5 (transient) -> 5.
    // (Measured: 10 / 8 instead of 5 / 4 iterations per pass, cfg 3 MIXED 1.3146-1.3165 -> 1.3128 s, FP64 1.3543-1.3550 ->
    // 1.3497 s.)
    const int period = opts->true_resid_period > 0 ? opts->true_resid_period : 20;
    P.unroll = 4;
    for (int u : {10, 8, 6, 5, 4, 3})
      if (period % u == 0) { P.unroll = u; break; }
  }
  P.k2blocks = k2_blocks(L.n);
  if (cheb && cheb_pairs_tma(L, code, T)) {
    P.pair_tma = 1;
    P.dia = dia_D; P.tnx = L.nx; P.tny = L.ny;
    P.tocc = pair_tma_occupancy(T) * 100 + pair_tma_rows(L, T);
  }
  cudaGetDevice(&P.device);
  return P;
}

static int solve_common(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, const double* b_D,
                        const double* power_D, double* x_D, void* work_D, size_t work_bytes,
                        cuth_result_t* result_D, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  rc = check_opts(opts);
  if (rc) return rc;
  if (!dia_D || !x_D || !work_D || !result_D || (!b_D && !power_D)) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || !aligned16(x_D) || !aligned16(work_D) || !aligned16(b_D) || !aligned16(power_D) ||
      ((uintptr_t)result_D & 7u))
    return CUTH_ERR_ALIGN;
  const bool transient = power_D != nullptr;
  if (transient && !(grid->cvol_H && grid->dt > 0.0)) return CUTH_ERR_NOT_TRANSIENT;
  if (work_bytes < cuth_workspace_bytes(grid, opts)) return CUTH_ERR_SIZE;
  cudaStream_t st = (cudaStream_t)stream;
  const bool cheb = opts->preconditioner == CUTH_PRECOND_CHEBYSHEV;
  const bool with_b = grid->cvol_H && grid->dt > 0.0;
  Tune T;
  make_tune(&opts->tuning, &T);
  if (opts->precision == CUTH_MIXED_STD32) T.traversal = 1;    // the ablation operator exists in the flat kernels only
  if (opts->precision == CUTH_FIXED32) T.traversal = 1;
  Workspace w = carve_workspace(work_D, L.n, with_b, cheb);
  DiaDev A = dev_view(dia_D, L, T);
  const int blocks = grid_blocks(L.n);
  if (transient) {
    k_transient_rhs<<<blocks, kThreads, 0, st>>>(A, power_D, x_D, w.b);
    CU(cudaGetLastError());
  }
  Ctx c;
  memset(&c, 0, sizeof c);
  c.A = A;
  c.b = transient ? w.b : b_D;
  c.x = x_D; c.r = w.r; c.p = w.p; c.p2 = w.p2; c.mu = w.mu;
  c.result = result_D;
  c.rtol = opts->rtol;
  c.precision = opts->precision;
  c.max_iters = opts->max_iters;
  c.period = opts->true_resid_period > 0 ? opts->true_resid_period : 20;
  c.jacobi = opts->preconditioner == CUTH_PRECOND_JACOBI ? 1 : 0;
  c.cheb = 0;
  if (cheb) fill_cheb(&c, opts, w);
  c.early_op = opts->precision == CUTH_MIXED_STD32 ? OP_STD32 : OP_DIFF32;
  c.transient_call = transient ? 1 : 0;
  c.k1_split = (use_zmarch(L, T) && k1_thin_stack(L, T, opts) == 2) ? 1 : 0;
  // persistent kernel: phases A and B in one on the smallest grids (not with the ablation operator)
  c.persist_fuse = (L.n <= (1 << 14) && c.early_op == OP_DIFF32) ? 1 : 0;
  c.soft_restart = 1;         // promotion keeps p while the drift is small (DESIGN.md R-G11)
  c.soft_drift2 = 1e-2;       // ||t - r|| <= 0.1 ||t||
  k_set_ctx<<<1, 32, 0, st>>>(c, w.ctx, w.ctl);
  CU(cudaGetLastError());
  { std::lock_guard<std::mutex> lk(g_mu); g_last_dia[work_D] = dia_D; }
  if (opts->precision == CUTH_FIXED32) {       // ablation: the paper's fixed-FP32 solver, one cooperative kernel
    int nb = coresident_blocks(3, (const void*)k_pcg_fixed32, 1, kPersistMaxBlocks, 0, kPersistMaxThreads);
    if (nb > 128) nb = 128;
    if (nb <= 0) { g_last_err = "CUTH_FIXED32: cooperative launch unavailable"; return CUTH_ERR_CUDA; }
    Ctx* ctxp = w.ctx; Ctl* ctlp = w.ctl; double* part = w.partials;
    void* args[] = {&ctxp, &ctlp, &part};
    CU(cudaLaunchCooperativeKernel((void*)k_pcg_fixed32, dim3(nb), dim3(kPersistMaxThreads), args, 0, st));
    return CUTH_OK;
  }
  if (use_cluster(L, opts, T)) {
    const cudaError_t e = launch_cluster(L, w.ctx, w.ctl, 1, st, T.loop_mode != 4);
    if (e == cudaSuccess) return CUTH_OK;
    if (T.loop_mode >= 3) return cuda_fail(e, "cudaLaunchKernelExC(k_pcg_cluster)");
    // automatic mode: fall through to the persistent kernel / the graph
  } else if (T.loop_mode >= 3) {
    g_last_err = "loop_mode 3 / 4: the grid does not fit one cluster, or the options are not served by the cluster kernel";
    return CUTH_ERR_VALUE;
  }
  if (use_persistent(L, cheb, T)) {
    Ctx* ctxp = w.ctx; Ctl* ctlp = w.ctl; double* part = w.partials;
    void* args[] = {&ctxp, &ctlp, &part};
    const PersistConfig pc = persistent_config(L.n);
    const cudaError_t e = cudaLaunchCooperativeKernel((void*)k_pcg_persistent, dim3(pc.blocks), dim3(pc.threads), args, 0, st);
    if (e == cudaSuccess) return CUTH_OK;
    if (T.loop_mode == 2) return cuda_fail(e, "cudaLaunchCooperativeKernel(k_pcg_persistent)");
    cudaGetLastError();       // automatic mode: the graph loop serves every grid (e.g. under an SM-limited context)
  }
  cudaGraphExec_t ex;
  rc = get_graph(w, work_D, make_plan(L, T, opts, with_b, dia_D), L, T, &ex);
  if (rc) return rc;
  CU(cudaGraphLaunch(ex, st));
  return CUTH_OK;
}


// Extreme eigenvalues of the symmetric tridiagonal T (diagonal a[0..m), off-diagonal b[0..m-1)) by Sturm
// bisection in fp64 on the host ("the solution of the spectrum of T is executed on CPUs").
static int sturm_count(const double* a, const double* b, int m, double x) {   // #eigenvalues < x
  int cnt = 0;
  double q = a[0] - x;
  if (q < 0) ++cnt;
  for (int i = 1; i < m; ++i) {
    if (q == 0.0) q = 1e-300;
    q = a[i] - x - b[i - 1] * b[i - 1] / q;
    if (q < 0) ++cnt;
  }
  return cnt;
}
static void tridiag_extremes(const double* a, const double* b, int m, double* lo, double* hi) {
  double gl = a[0], gu = a[0];
  for (int i = 0; i < m; ++i) {
    const double r = (i > 0 ? fabs(b[i - 1]) : 0.0) + (i + 1 < m ? fabs(b[i]) : 0.0);
    gl = fmin(gl, a[i] - r); gu = fmax(gu, a[i] + r);
  }
  for (int which = 0; which < 2; ++which) {
    const int target = which == 0 ? 1 : m;          // smallest: count(x) >= 1; largest: count(x) >= m
    double l = gl, u = gu;
    for (int it = 0; it < 200 && u - l > 1e-15 * fmax(fabs(l), fabs(u)); ++it) {
      const double mid = 0.5 * (l + u);
      if (sturm_count(a, b, m, mid) >= target) u = mid; else l = mid;
    }
    *(which == 0 ? lo : hi) = 0.5 * (l + u);
  }
}

}  // namespace cuth

using namespace cuth;

extern "C" {

size_t cuth_dia_bytes(const cuth_grid_t* grid) {
  DiaLayout L;
  if (!make_layout(grid, &L)) return 0;
  return L.bytes;
}

size_t cuth_workspace_bytes(const cuth_grid_t* grid, const cuth_opts_t* opts) {
  DiaLayout L;
  if (!make_layout(grid, &L)) return 0;
  return carve_workspace(nullptr, L.n, grid->cvol_H && grid->dt > 0.0,
                         opts && opts->preconditioner == CUTH_PRECOND_CHEBYSHEV).bytes;
}

int cuth_build_dia(const cuth_grid_t* grid, void* dia_D, size_t dia_bytes, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!dia_D || !grid->dz_H || !grid->kappa_D) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || ((uintptr_t)grid->kappa_D & 7u)) return CUTH_ERR_ALIGN;
  if (dia_bytes < L.bytes) return CUTH_ERR_SIZE;
  for (int64_t z = 0; z < grid->nz; ++z) {
    if (!(grid->dz_H[z] > 0.0)) return CUTH_ERR_VALUE;
    if (grid->cvol_H && grid->dt > 0.0 && !(grid->cvol_H[z] > 0.0)) return CUTH_ERR_VALUE;
  }
  cudaError_t e = cudaSuccess;
  rc = launch_build(grid, L, dia_D, (cudaStream_t)stream, &e);
  if (rc == CUTH_ERR_CUDA) return cuda_fail(e, "cuth_build_dia");
  return rc;
}

int cuth_import_csr(const cuth_grid_t* grid, const int64_t* rowptr_D, const int32_t* col_D, const double* val_D,
                    const double* rowsum_layer_H, void* dia_D, size_t dia_bytes, cuth_import_report_t* report_H,
                    void* stream) {
  return cuth_import_csr_n(grid, rowptr_D, col_D, val_D, -1, rowsum_layer_H, dia_D, dia_bytes, report_H, stream);
}

int cuth_import_csr_n(const cuth_grid_t* grid, const int64_t* rowptr_D, const int32_t* col_D, const double* val_D,
                      int64_t nnz, const double* rowsum_layer_H, void* dia_D, size_t dia_bytes,
                      cuth_import_report_t* report_H, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!dia_D || !rowptr_D || !col_D || !val_D) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || ((uintptr_t)rowptr_D & 7u) || ((uintptr_t)col_D & 3u) || ((uintptr_t)val_D & 7u))
    return CUTH_ERR_ALIGN;
  if (dia_bytes < L.bytes) return CUTH_ERR_SIZE;
  if (rowsum_layer_H)
    for (int64_t z = 0; z < grid->nz; ++z)
      if (!(rowsum_layer_H[z] >= 0.0) || std::isinf(rowsum_layer_H[z])) return CUTH_ERR_VALUE;
  cuth_import_report_t rep;
  memset(&rep, 0, sizeof rep);
  cudaError_t e = cudaSuccess;
  rc = launch_import(grid, L, rowptr_D, col_D, val_D, rowsum_layer_H, dia_D, &rep, (cudaStream_t)stream, &e, nullptr,
                     nnz < 0 ? -1 : nnz);
  if (report_H) *report_H = rep;
  if (rc == CUTH_ERR_CUDA) return cuda_fail(e, "cuth_import_csr");
  return rc;
}

int cuth_dia_view(const void* dia_D, const cuth_grid_t* grid, const double** vals_D, const float** vals32_D,
                  const double** inv_diag_D, int64_t ptr_H[5], int64_t off_H[4]) {
  DiaLayout L;
  if (!dia_D) return CUTH_ERR_NULL;
  if (!make_layout(grid, &L)) return grid ? CUTH_ERR_DIMS : CUTH_ERR_NULL;
  const char* base = (const char*)dia_D;
  if (vals_D) *vals_D = (const double*)(base + L.o_vals);
  if (vals32_D) *vals32_D = (const float*)(base + L.o_vals32);
  if (inv_diag_D) *inv_diag_D = (const double*)(base + L.o_dinv);
  if (ptr_H) for (int k = 0; k < 5; ++k) ptr_H[k] = L.ptr[k];
  if (off_H) for (int k = 0; k < 4; ++k) off_H[k] = L.off[k];
  return CUTH_OK;
}

}  // extern "C"

// cuth_spmv with TMA-staged operands (cuth_spmv_tma.cuh): wherever the two-column z-marching kernel would run, nx % 4 == 0
// (strides of the tensor maps), the plane has at least one resident wave of 64 x 8 tiles and the stack at least 12
// layers; k1_variant 1 / 3 keep the LDG kernels, 2 forces it.  The kernel is persistent over tiles: as many CTAs as give every CTA the same number of
// tiles (cfg 3: 2048 tiles, 592 resident -> 4 waves -> 512 CTAs of exactly 4 tiles).
template <bool MIXED>
static int spmv_tma_blocks(const DiaLayout& L) {
  const void* fn = (const void*)k_spmv_tma<MIXED>;
  static_assert(sizeof(SpSmem<MIXED>) <= 227 * 1024, "stages of the TMA SpMV");
  cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SpSmem<MIXED>));
  const int resident = coresident_blocks(MIXED ? 5 : 6, fn, MIXED ? 4 : 2, kMaxBlocks, sizeof(SpSmem<MIXED>));
  if (resident <= 0) return 0;
  const int64_t tiles = ((L.nx + K1X - 1) / K1X) * ((L.ny + K1Y - 1) / K1Y);
  const int64_t waves = (tiles + resident - 1) / resident;
  return (int)((tiles + waves - 1) / waves);
}
static bool spmv_tma(const DiaLayout& L, const Tune& T) {
  if (!use_zmarch(L, T) || !zmarch_x2(L, T) || T.k1_variant == 3) return false;
  if ((L.nx % 4) != 0 || encode_tiled_fn() == nullptr) return false;
  if (T.k1_variant == 2) return true;
  // Measured on B200, TMA / LDG: cfg 3 (nz = 16) fp64 0.126 / 0.133 ms, fp32-stored 0.078 / 0.086 ms; cfg 4 (nz = 8: nine
  // steps for eight planes) fp64 0.977 / 0.981 ms, fp32-stored 0.714 / 0.637 ms -- so thin stacks keep the LDG kernel.
  return ((L.nx + K1X - 1) / K1X) * ((L.ny + K1Y - 1) / K1Y) >= 592 && L.nz >= 12;
}
template <bool MIXED>
static cudaError_t launch_spmv_tma(const DiaLayout& L, const DiaDev& A, const void* dia_D, const double* x_D, double* y_D,
                                   cudaStream_t st) {
  using ST = SpStage<MIXED>;
  const int blocks = spmv_tma_blocks<MIXED>(L);
  if (blocks <= 0) return cudaErrorInvalidConfiguration;
  const char* base = (const char*)dia_D;
  CUtensorMap tx, td, t1, t2, t3;
  bool ok = make_map3d(&tx, x_D, 8, L, K1VW, K1VH) && make_map3d(&td, A.d0, 8, L, K1X, K1Y);
  if (MIXED)
    ok = ok && make_map3d(&t1, A.f1, 4, L, ST::W1, K1Y) && make_map3d(&t2, A.f2, 4, L, K1X, K1Y + 1) &&
         make_map3d(&t3, A.f3, 4, L, K1X, K1Y);
  else
    ok = ok && make_map3d(&t1, base + L.o_f64a, 8, L, ST::W1, K1Y) &&
         make_map3d(&t2, base + L.o_f64a + L.f64a_stride, 8, L, K1X, K1Y + 1) &&
         make_map3d(&t3, base + L.o_f64a + 2 * L.f64a_stride, 8, L, K1X, K1Y);
  if (!ok) return cudaErrorInvalidValue;
  k_spmv_tma<MIXED><<<blocks, kThreads, sizeof(SpSmem<MIXED>), st>>>(A, y_D, tx, td, t1, t2, t3);
  return cudaGetLastError();
}

extern "C" {

int cuth_spmv_tuned(const void* dia_D, const cuth_grid_t* grid, int precision, const cuth_tuning_t* tuning,
                    const double* x_D, double* y_D, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!dia_D || !x_D || !y_D) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || !aligned16(x_D) || !aligned16(y_D)) return CUTH_ERR_ALIGN;
  if (precision != CUTH_FP64 && precision != CUTH_MIXED && precision != CUTH_MIXED_STD32) return CUTH_ERR_VALUE;
  if (x_D == y_D) return CUTH_ERR_VALUE;
  Tune T;
  if (make_tune(tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  if (precision == CUTH_MIXED_STD32) T.traversal = 1;
  DiaDev A = dev_view(dia_D, L, T);
  const int sb = stencil_blocks(L, T);
  const int blocks = sb > 0 ? sb : grid_blocks(L.n);
  cudaStream_t st = (cudaStream_t)stream;
  if (precision != CUTH_MIXED_STD32 && spmv_tma(L, T)) {
    const cudaError_t e = precision == CUTH_MIXED ? launch_spmv_tma<true>(L, A, dia_D, x_D, y_D, st)
                                                  : launch_spmv_tma<false>(L, A, dia_D, x_D, y_D, st);
    if (e == cudaSuccess) return CUTH_OK;
    if (T.k1_variant == 2) return cuda_fail(e, "k_spmv_tma");
    cudaGetLastError();                       // automatic: the LDG kernel serves every grid
  }
  if (precision == CUTH_MIXED_STD32) k_spmv_only<OP_STD32><<<blocks, kThreads, 0, st>>>(A, x_D, y_D);
  else if (precision == CUTH_MIXED) k_spmv_only<OP_DIFF32><<<blocks, kThreads, 0, st>>>(A, x_D, y_D);
  else k_spmv_only<OP_FP64><<<blocks, kThreads, 0, st>>>(A, x_D, y_D);
  CU(cudaGetLastError());
  return CUTH_OK;
}

int cuth_spmv(const void* dia_D, const cuth_grid_t* grid, int precision, const double* x_D, double* y_D,
              void* stream) {
  return cuth_spmv_tuned(dia_D, grid, precision, nullptr, x_D, y_D, stream);
}

int cuth_pcg_solve(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, const double* b_D,
                   double* x_D, void* work_D, size_t work_bytes, cuth_result_t* result_D, void* stream) {
  if (!b_D) return CUTH_ERR_NULL;
  return solve_common(dia_D, grid, opts, b_D, nullptr, x_D, work_D, work_bytes, result_D, stream);
}

int cuth_import_coo(const cuth_grid_t* grid, const int32_t* row_D, const int32_t* col_D, const double* val_D, int64_t nnz,
                    const double* rowsum_layer_H, void* dia_D, size_t dia_bytes, cuth_import_report_t* report_H,
                    void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!dia_D || !row_D || !col_D || !val_D) return CUTH_ERR_NULL;
  if (nnz < 0) return CUTH_ERR_VALUE;
  if (!aligned16(dia_D) || ((uintptr_t)row_D & 3u) || ((uintptr_t)col_D & 3u) || ((uintptr_t)val_D & 7u))
    return CUTH_ERR_ALIGN;
  if (dia_bytes < L.bytes) return CUTH_ERR_SIZE;
  if (rowsum_layer_H)
    for (int64_t z = 0; z < grid->nz; ++z)
      if (!(rowsum_layer_H[z] >= 0.0) || std::isinf(rowsum_layer_H[z])) return CUTH_ERR_VALUE;
  cuth_import_report_t rep;
  memset(&rep, 0, sizeof rep);
  cudaError_t e = cudaSuccess;
  rc = launch_import(grid, L, nullptr, col_D, val_D, rowsum_layer_H, dia_D, &rep, (cudaStream_t)stream, &e, row_D, nnz);
  if (report_H) *report_H = rep;
  if (rc == CUTH_ERR_CUDA) return cuda_fail(e, "cuth_import_coo");
  return rc;
}

size_t cuth_batch_workspace_bytes(const cuth_grid_t* grid, int nrhs) {
  DiaLayout L;
  if (!make_layout(grid, &L) || nrhs < 1 || nrhs > kBatchMaxRhs) return 0;
  return carve_batch_workspace(nullptr, L.n, nrhs).bytes;
}

int cuth_pcg_solve_batch(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, int nrhs,
                         const double* b_D, double* x_D, void* work_D, size_t work_bytes, cuth_result_t* result_D,
                         void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  rc = check_opts(opts);
  if (rc) return rc;
  if (nrhs < 1 || nrhs > kBatchMaxRhs) return CUTH_ERR_VALUE;
  if (opts->preconditioner != CUTH_PRECOND_JACOBI && opts->preconditioner != CUTH_PRECOND_NONE) return CUTH_ERR_VALUE;
  if (opts->precision != CUTH_FP64 && opts->precision != CUTH_MIXED) return CUTH_ERR_VALUE;
  if (!dia_D || !b_D || !x_D || !work_D || !result_D) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || !aligned16(x_D) || !aligned16(work_D) || !aligned16(b_D) || ((uintptr_t)result_D & 7u))
    return CUTH_ERR_ALIGN;
  BatchWorkspace w = carve_batch_workspace(work_D, L.n, nrhs);
  if (work_bytes < w.bytes) return CUTH_ERR_SIZE;
  cudaStream_t st = (cudaStream_t)stream;
  Tune T;
  make_tune(&opts->tuning, &T);
  if (use_cluster(L, opts, T)) {
    // Small grids: ONE CLUSTER PER RIGHT-HAND SIDE (cuth_cluster.cuh) -- each solve is exactly cuth_pcg_solve's, the
    // clusters run side by side on the 148 SMs (18 at a time with 8 CTAs each).  cfg 1, 32 right-hand sides: 4.7 ms in the
    // lock-step kernel below, 2.6 ms here.  The per-solve contexts live in the partials area of the batch workspace.
    static_assert(sizeof(Ctx) * kBatchMaxRhs <= sizeof(double) * 2 * 3 * (size_t)kBatchMaxRhs * kBatchMaxBlocks, "contexts fit");
    Ctx base;
    memset(&base, 0, sizeof base);
    base.A = dev_view(dia_D, L, T);
    base.b = b_D; base.x = x_D; base.result = result_D;
    base.rtol = opts->rtol; base.precision = opts->precision; base.max_iters = opts->max_iters;
    base.period = opts->true_resid_period > 0 ? opts->true_resid_period : 20;
    base.jacobi = opts->preconditioner == CUTH_PRECOND_JACOBI ? 1 : 0;
    base.early_op = OP_DIFF32;
    base.soft_restart = 1; base.soft_drift2 = 1e-2;
    Ctx* ctxs = reinterpret_cast<Ctx*>(w.partials);
    k_set_ctx_batch<<<1, kBatchMaxRhs, 0, st>>>(base, ctxs, w.ctl, nrhs);
    CU(cudaGetLastError());
    const cudaError_t e = launch_cluster(L, ctxs, w.ctl, nrhs, st, T.loop_mode != 4);
    if (e == cudaSuccess) return CUTH_OK;
    if (T.loop_mode >= 3) return cuda_fail(e, "cudaLaunchKernelExC(k_pcg_cluster, batch)");
  }
  // co-resident CTAs available, split into ceil(nrhs / S) chunks x ntiles row tiles
  const int max_blocks = coresident_blocks(1, (const void*)k_pcg_batch, 3, 1 << 20);
  const int nchunks = (nrhs + kBatchChunk - 1) / kBatchChunk;
  if (max_blocks < nchunks) { g_last_err = "cuth_pcg_solve_batch: cooperative launch unavailable"; return CUTH_ERR_CUDA; }
  const int64_t need = (L.n + (int64_t)kThreads - 1) / (int64_t)kThreads;
  int64_t ntiles = max_blocks / nchunks;
  if (ntiles > need) ntiles = need;
  // the barrier is fastest at >= 128 CTAs (see persistent_config): tiles beyond the rows only take part in it
  if (ntiles * nchunks < 128 && max_blocks >= 128) ntiles = (128 + nchunks - 1) / nchunks;
  if (ntiles > kBatchMaxBlocks) ntiles = kBatchMaxBlocks;
  BatchCtx c;
  memset(&c, 0, sizeof c);
  c.A = dev_view(dia_D, L, Tune());
  c.b = b_D; c.x = x_D; c.r = w.r; c.p = w.p; c.mu = w.mu;
  c.result = result_D;
  c.rtol = opts->rtol;
  c.nrhs = nrhs; c.max_iters = opts->max_iters;
  c.jacobi = opts->preconditioner == CUTH_PRECOND_JACOBI ? 1 : 0;
  c.ntiles = (int32_t)ntiles;
  c.precision = opts->precision;
  c.period = opts->true_resid_period > 0 ? opts->true_resid_period : 20;
  k_batch_set_ctx<<<1, 32, 0, st>>>(c, w.ctx, w.ctl);
  CU(cudaGetLastError());
  BatchCtx* ctxp = w.ctx; Ctl* ctlp = w.ctl; double* part = w.partials;
  void* args[] = {&ctxp, &ctlp, &part};
  CU(cudaLaunchCooperativeKernel((void*)k_pcg_batch, dim3((unsigned)(ntiles * nchunks)), dim3(kThreads), args, 0, st));
  return CUTH_OK;
}

int cuth_transient_step(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts,
                        const double* power_D, double* T_D, void* work_D, size_t work_bytes,
                        cuth_result_t* result_D, void* stream) {
  if (!power_D) return CUTH_ERR_NULL;
  return solve_common(dia_D, grid, opts, nullptr, power_D, T_D, work_D, work_bytes, result_D, stream);
}

int cuth_profile_kernel(void* work_D, const cuth_grid_t* grid, const cuth_opts_t* opts, int kernel_id, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!work_D || !opts) return CUTH_ERR_NULL;
  Tune T;
  if (make_tune(&opts->tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  if (opts->precision == CUTH_MIXED_STD32) T.traversal = 1;
  cudaStream_t st = (cudaStream_t)stream;
  const bool with_b = grid->cvol_H && grid->dt > 0.0;
  Workspace w = carve_workspace(work_D, L.n, with_b);
  const int blocks = grid_blocks(L.n);
  const int sb = stencil_blocks(L, T) > 0 ? stencil_blocks(L, T) : blocks;
  cudaGraphConditionalHandle h0 = 0;
  switch (kernel_id) {
    case -1: k_mark_no_graph<<<1, 1, 0, st>>>(w.ctl, 0); break;
    case -2: k_mark_no_graph<<<1, 1, 0, st>>>(w.ctl, 1); break;
    case 0: k_pupdate<<<blocks, kThreads, 0, st>>>(w.ctx, w.ctl); break;
    case 1: k_spmv_dot<<<sb, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials); break;
    case 2: k_update<true><<<blocks, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials, h0, h0); break;
    case 4:
      if (fused_tma(L, T, opts->preconditioner == CUTH_PRECOND_CHEBYSHEV) && k1_thin_stack(L, T, opts) != 1) {
        const void* dia = nullptr;
        { std::lock_guard<std::mutex> lk(g_mu);
          auto it = g_last_dia.find(work_D);
          if (it != g_last_dia.end()) dia = it->second; }
        if (!dia) return CUTH_ERR_VALUE;           // no solve has used this workspace yet
        K1Maps km, km64;
        if (!make_k1_maps(&km, &km64, L, dia, w)) return CUTH_ERR_CUDA;
        Ctx* ctxp = w.ctx; Ctl* ctlp = w.ctl; double* part = w.partials;
        void* a[] = {&ctxp, &ctlp, &part, &km.z, &km.p, &km.p2, &km.d, &km64.d, &km.m1, &km.m2, &km.m3,
                     &km64.m1, &km64.m2, &km64.m3};
        CU(cudaLaunchKernel((const void*)k_fused_pspmv_tma, dim3(fused_tma_blocks(L)), dim3(kThreads), a,
                            k1_tma_dyn_smem(), st));
        if (k1_thin_stack(L, T, opts) == 2)        // as in the graph: one of the two returns at once
          k_fused_pspmv_x2<<<fused_blocks(L, T), kThreads, 0, st>>>(w.ctx, w.ctl, w.partials);
      } else if (fused_x2(L, T)) k_fused_pspmv_x2<<<fused_blocks(L, T), kThreads, 0, st>>>(w.ctx, w.ctl, w.partials);
      else k_fused_pspmv<<<fused_blocks(L, T), kThreads, 0, st>>>(w.ctx, w.ctl, w.partials);
      break;
    case 5: k_update<false><<<k2_blocks(L.n), kK2Threads, 0, st>>>(w.ctx, w.ctl, w.partials, h0, h0); break;
    case 6: case 7: case 8: {      // one middle step of the Chebyshev apply: fp64 / fp32 on A2 / fp32 on A3 (fp16)
      const int code = kernel_id - 6;
      const bool x2 = code != 0 && cheb_x2(L, T);
      Ctx* ctxp = w.ctx; int step = 1, old = 1, cur = 0;
      void* args[] = {&ctxp, &step, &old, &cur};
      CU(cudaLaunchKernel(cheb_mid_fn(code, x2), dim3(x2 ? cheb_x2_blocks(L) : cheb_blocks(L, T)), dim3(kThreads), args, 0, st));
    } break;
    case 9: case 10: {            // one fused pair of Chebyshev passes, fp32 on A2 / on A3
      const void* dia = nullptr;
      { std::lock_guard<std::mutex> lk(g_mu);
        auto it = g_last_dia.find(work_D);
        if (it != g_last_dia.end()) dia = it->second; }
      if (!dia) return CUTH_ERR_VALUE;             // no solve has used this workspace yet
      const ChebOp op = {1, 1, 1, 0, 2, 3};
      const Workspace wc = carve_workspace(work_D, L.n, with_b, true);   // with the Z buffers
      CU(launch_pair(L, T, dia, wc, kernel_id == 10 ? 2 : 1, op, st));
    } break;
    case 3: k_true_resid<<<sb, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials, h0); break;
    default: return CUTH_ERR_VALUE;
  }
  CU(cudaGetLastError());
  return CUTH_OK;
}

int cuth_lanczos_bounds_tuned(const void* dia_D, const cuth_grid_t* grid, const cuth_tuning_t* tuning, const double* v0_D,
                              int steps, void* work_D, size_t work_bytes, double bounds_H[5], void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!dia_D || !v0_D || !work_D || !bounds_H) return CUTH_ERR_NULL;
  if (steps < 2 || steps > 120) return CUTH_ERR_VALUE;
  if (!aligned16(dia_D) || !aligned16(v0_D) || !aligned16(work_D)) return CUTH_ERR_ALIGN;
  Tune T;
  if (make_tune(tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  Workspace w = carve_workspace(work_D, L.n, grid->cvol_H && grid->dt > 0.0);
  if (work_bytes < w.bytes) return CUTH_ERR_SIZE;
  cudaStream_t st = (cudaStream_t)stream;
  DiaDev A = dev_view(dia_D, L, T);
  const int blocks = grid_blocks(L.n);
  const int sb = stencil_blocks(L, T) > 0 ? stencil_blocks(L, T) : blocks;
  LanczosScal* sc = (LanczosScal*)(w.partials + 3 * kMaxBlocks);
  static_assert(sizeof(LanczosScal) <= sizeof(double) * kMaxBlocks, "LanczosScal must fit one partial slot");
  CU(cudaMemsetAsync(sc, 0, sizeof(LanczosScal), st));
  if (T.lanczos_fp32) {
    // the paper's variant (PAPER.md:315 "matrix A2 is used", :340 "in FP32 precision using the fixed FP32 SpMV kernel"):
    // fp32 vectors in the same workspace buffers, A2 in standard form, fp32 arithmetic (flat traversal)
    float* u_cur = (float*)w.r; float* u_prev = (float*)w.p; float* t = (float*)w.mu;
    k_lanczos_init<float><<<blocks, kThreads, 0, st>>>(A, v0_D, u_cur, u_prev, sc, w.partials);
    for (int j = 0; j < steps; ++j) {
      k_lanczos_1_f32<<<blocks, kThreads, 0, st>>>(A, u_cur, u_prev, t, sc, w.partials);
      k_lanczos_2<float><<<blocks, kThreads, 0, st>>>(L.n, u_cur, t, u_prev, sc, w.partials);
      float* tmp = u_prev; u_prev = u_cur; u_cur = tmp;
    }
  } else {
    double* u_cur = w.r; double* u_prev = w.p; double* t = w.mu;
    k_lanczos_init<double><<<blocks, kThreads, 0, st>>>(A, v0_D, u_cur, u_prev, sc, w.partials);
    for (int j = 0; j < steps; ++j) {
      k_lanczos_1<<<sb, kThreads, 0, st>>>(A, u_cur, u_prev, t, sc, w.partials);
      k_lanczos_2<double><<<blocks, kThreads, 0, st>>>(L.n, u_cur, t, u_prev, sc, w.partials);
      double* tmp = u_prev; u_prev = u_cur; u_cur = tmp;     // u_{j+1} was written over u_{j-1}
    }
  }
  CU(cudaGetLastError());
  LanczosScal h;
  CU(cudaMemcpyAsync(&h, sc, sizeof h, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  int m = steps;
  for (int j = 0; j < steps; ++j)
    if (!(h.out_beta[j] > 0.0) || !(h.out_alpha[j] == h.out_alpha[j])) { m = j + 1; break; }   // invariant subspace
  tridiag_extremes(h.out_alpha, h.out_beta, m, &bounds_H[0], &bounds_H[1]);
  bounds_H[2] = h.out_beta[127];       // Gershgorin bound (k_lanczos_init)
  // Interval handed to Alg. 3 (DESIGN.md R-C2): alpha = smallest Ritz value; beta = 1.05 x the largest Ritz
  // value (Ritz values approach lambda_max from below), never above the Gershgorin bound.
  bounds_H[3] = bounds_H[0];
  bounds_H[4] = fmin(1.05 * bounds_H[1], bounds_H[2]);
  return CUTH_OK;
}

int cuth_lanczos_bounds(const void* dia_D, const cuth_grid_t* grid, const double* v0_D, int steps, void* work_D,
                        size_t work_bytes, double bounds_H[5], void* stream) {
  return cuth_lanczos_bounds_tuned(dia_D, grid, nullptr, v0_D, steps, work_D, work_bytes, bounds_H, stream);
}

int cuth_cheb_apply(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, const double* r_D,
                    double* z_D, void* work_D, size_t work_bytes, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  rc = check_opts(opts);
  if (rc) return rc;
  if (opts->preconditioner != CUTH_PRECOND_CHEBYSHEV) return CUTH_ERR_VALUE;
  if (opts->precision != CUTH_FP64 && opts->precision != CUTH_MIXED) return CUTH_ERR_VALUE;
  if (!dia_D || !r_D || !z_D || !work_D) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || !aligned16(r_D) || !aligned16(z_D) || !aligned16(work_D)) return CUTH_ERR_ALIGN;
  if (work_bytes < cuth_workspace_bytes(grid, opts)) return CUTH_ERR_SIZE;
  Tune T;
  make_tune(&opts->tuning, &T);
  cudaStream_t st = (cudaStream_t)stream;
  Workspace w = carve_workspace(work_D, L.n, grid->cvol_H && grid->dt > 0.0, true);
  Ctx c;
  memset(&c, 0, sizeof c);
  c.A = dev_view(dia_D, L, T);
  c.r = const_cast<double*>(r_D);      // read only here
  fill_cheb(&c, opts, w);
  c.cz = z_D;
  k_set_ctx<<<1, 32, 0, st>>>(c, w.ctx, w.ctl);
  CU(cudaGetLastError());
  const int sb = cheb_blocks(L, T);
  const int k = opts->cheb_degree;
  const int code = cheb_code(opts);
  const bool x2 = code != 0 && cheb_x2(L, T);
  Ctx* ctxp = w.ctx; Ctl* ctlp = w.ctl; double* part = w.partials;
  { void* a[] = {&ctxp};
    CU(cudaLaunchKernel(cheb_first_fn(code), dim3(sb), dim3(kThreads), a, 0, st)); }
  for (const ChebOp& op : cheb_schedule(k, cheb_pairs(L, code, T), cheb_pairs_tma(L, code, T))) {
    int step = op.step, old = op.old, cur = op.cur;
    if (op.kind == 1 || op.kind == 3) {
      CU(launch_pair(L, T, dia_D, w, code, op, st));
    } else if (op.kind == 0) {
      void* a[] = {&ctxp, &step, &old, &cur};
      CU(cudaLaunchKernel(cheb_mid_fn(code, x2), dim3(x2 ? cheb_x2_blocks(L) : sb), dim3(kThreads), a, 0, st));
    } else {
      void* a[] = {&ctxp, &ctlp, &part, &step, &old, &cur};
      CU(cudaLaunchKernel(cheb_last_fn(code), dim3(sb), dim3(kThreads), a, 0, st));
    }
  }
  CU(cudaGetLastError());
  return CUTH_OK;
}

// Test hook: the decision function of the solver kernels on caller-given scalars (include/cuth.h).
__global__ void k_policy_probe(double rr, double tt, double dd, double tt_prev, double rr_prev, double bb, double rtol,
                               double soft_drift, int flags, int32_t* out) {
  Ctl ctl;
  memset(&ctl, 0, sizeof ctl);
  Ctx c;
  memset(&c, 0, sizeof c);
  c.rtol = rtol; c.max_iters = 1000; c.soft_restart = soft_drift >= 0.0 ? 1 : 0;
  c.soft_drift2 = soft_drift > 0.0 ? soft_drift * soft_drift : 1e-2;
  ctl.status = CUTH_SOLVE_RUNNING;
  ctl.bb = bb; ctl.tol2 = rtol * rtol * bb; ctl.sw2 = fmax(rtol, rtol * rtol) * bb;
  ctl.rr = rr; ctl.tt_prev = tt_prev; ctl.rr_prev_eval = rr_prev;
  ctl.stage = (flags & 1) ? 1 : 0;
  ctl.conv_rec = (flags & 2) ? 1 : 0;
  ctl.it = (flags & 4) ? c.max_iters : 10;
  const unsigned go = policy_after_true(&ctl, c, tt, dd);
  out[0] = (int32_t)go; out[1] = ctl.stage; out[2] = ctl.switch_reason; out[3] = ctl.switch_mask; out[4] = ctl.restart;
  out[5] = ctl.status; out[6] = ctl.promotions; out[7] = 0;
}

int cuth_policy_probe(const double in_H[8], int flags, int32_t* out_D, void* stream) {
  if (!in_H || !out_D) return CUTH_ERR_NULL;
  if (((uintptr_t)out_D & 3u)) return CUTH_ERR_ALIGN;
  k_policy_probe<<<1, 1, 0, (cudaStream_t)stream>>>(in_H[0], in_H[1], in_H[2], in_H[3], in_H[4], in_H[5], in_H[6], in_H[7],
                                                    flags, out_D);
  CU(cudaGetLastError());
  return CUTH_OK;
}

int cuth_tridiag_extremes(const double* alpha_H, const double* beta_H, int m, double out_H[2]) {
  if (!alpha_H || !out_H || (m > 1 && !beta_H)) return CUTH_ERR_NULL;
  if (m < 1) return CUTH_ERR_VALUE;
  tridiag_extremes(alpha_H, beta_H, m, &out_H[0], &out_H[1]);
  return CUTH_OK;
}

int cuth_release_workspace(const void* work_D) {
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_graphs.find(work_D);
  if (it != g_graphs.end()) {
    cudaGraphExecDestroy(it->second.exec);
    cudaGraphDestroy(it->second.graph);
    g_graphs.erase(it);
  }
  g_last_dia.erase(work_D);
  return CUTH_OK;
}

const char* cuth_last_cuda_error(void) { return g_last_err.c_str(); }

int cuth_version(void) { return 10000; }

int cuth_launches_per_iteration(const cuth_grid_t* grid, const cuth_opts_t* opts) {
  DiaLayout L;
  Tune T;
  if (!make_layout(grid, &L) || !opts || make_tune(&opts->tuning, &T) != CUTH_OK) return 0;
  if (opts->precision == CUTH_MIXED_STD32) T.traversal = 1;
  if (use_cluster(L, opts, T)) return 0;                                                   // one cluster-resident kernel
  if (use_persistent(L, opts->preconditioner == CUTH_PRECOND_CHEBYSHEV, T)) return 0;      // one persistent kernel for the whole solve
  if (!use_zmarch(L, T)) return 3;
  return k1_thin_stack(L, T, opts) == 2 ? 3 : 2;   // thin stacks, MIXED: K1 is two nodes, one of which returns at once
}

int cuth_traversal(const cuth_grid_t* grid, const cuth_opts_t* opts) {
  DiaLayout L;
  Tune T;
  if (!opts) return CUTH_ERR_NULL;
  if (!make_layout(grid, &L)) return CUTH_ERR_DIMS;
  if (check_opts(opts) != CUTH_OK || make_tune(&opts->tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  if (opts->precision == CUTH_MIXED_STD32 || opts->precision == CUTH_FIXED32) T.traversal = 1;
  return use_zmarch(L, T) ? 2 : 1;
}

int cuth_loop_home(const cuth_grid_t* grid, const cuth_opts_t* opts) {
  DiaLayout L;
  Tune T;
  if (!opts) return CUTH_ERR_NULL;
  if (!make_layout(grid, &L)) return CUTH_ERR_DIMS;
  if (check_opts(opts) != CUTH_OK || make_tune(&opts->tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  if (opts->precision == CUTH_FIXED32) return 4;
  if (opts->precision == CUTH_MIXED_STD32) T.traversal = 1;
  if (use_cluster(L, opts, T)) return 3;
  if (T.loop_mode >= 3) return CUTH_ERR_VALUE;
  return use_persistent(L, opts->preconditioner == CUTH_PRECOND_CHEBYSHEV, T) ? 2 : 1;
}

int cuth_cheb_launches(const cuth_grid_t* grid, const cuth_opts_t* opts, int* pairs_out) {
  DiaLayout L;
  if (!opts) return CUTH_ERR_NULL;
  if (!make_layout(grid, &L)) return CUTH_ERR_DIMS;
  if (opts->preconditioner != CUTH_PRECOND_CHEBYSHEV) { if (pairs_out) *pairs_out = 0; return 0; }
  Tune T;
  if (make_tune(&opts->tuning, &T) != CUTH_OK) return CUTH_ERR_VALUE;
  int pairs = 0, launches = 1;                   // FIRST
  for (const ChebOp& op : cheb_schedule(opts->cheb_degree, cheb_pairs(L, cheb_code(opts), T),
                                        cheb_pairs_tma(L, cheb_code(opts), T))) {
    ++launches;
    if (op.kind == 1 || op.kind == 3) ++pairs;
  }
  if (pairs_out) *pairs_out = pairs;
  return launches;
}

}  // extern "C"
