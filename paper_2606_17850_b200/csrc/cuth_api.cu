// cuth_api.cu -- the C ABI of include/cuth.h: argument checks, CUDA-graph construction, launches.
// The PCG loop is ONE CUDA graph per workspace.  Nothing in it synchronises with the host.
//   small planes (flat traversal):  k_init -> WHILE{ k_pupdate, k_spmv_dot, k_update<x>,
//                                   IF{ k_true_resid, k_restart } } -> k_finalize
//   large planes (fused path):      k_init -> WHILE{ k_fused_pspmv, k_update<no x>,
//                                   IF{ k_flush_x, k_true_resid, k_restart } } -> k_finalize
#include <cmath>
#include <cstdio>
#include <atomic>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <unordered_map>

#include "cuth_fused.cuh"

namespace cuth {

int launch_build(const cuth_grid_t* g, const DiaLayout& L, void* dia_D, cudaStream_t st, cudaError_t* err);

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

static int check_grid(const cuth_grid_t* g, DiaLayout* L) {
  if (!g) return CUTH_ERR_NULL;
  if (!make_layout(g, L)) return CUTH_ERR_DIMS;
  if (!(g->dx > 0.0) || !(g->dy > 0.0) || !(g->h_top >= 0.0)) return CUTH_ERR_VALUE;
  return CUTH_OK;
}

static std::atomic<int> g_traversal{0};   // 0 auto, 1 flat, 2 z-march (cuth_set_traversal)

// Traversal choice: the flat kernel relies on L2 to keep the +-nx*ny neighbours (two planes of six
// arrays, 96 B per plane cell); beyond ~1/3 of the 126 MB L2 that fails and z-marching wins.
static bool use_zmarch(const DiaLayout& L) {
  const int mode = g_traversal.load();
  if (mode == 1) return false;
  if (mode == 2) return true;
  return L.nxny >= (1 << 18);
}

static int stencil_blocks(const DiaLayout& L) {
  if (!use_zmarch(L)) return -1;
  const int64_t tiles = ((L.nx + ZTX - 1) / ZTX) * ((L.ny + ZTY - 1) / ZTY);
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}

static int fused_blocks(const DiaLayout& L) {
  const int64_t tiles = ((L.nx + FTX - 1) / FTX) * ((L.ny + FTY - 1) / FTY);
  return (int)(tiles < kMaxBlocks ? tiles : kMaxBlocks);
}

static DiaDev dev_view(const void* dia_D, const DiaLayout& L) {
  const char* base = (const char*)dia_D;
  const double* v = (const double*)(base + L.o_vals);
  const float* f = (const float*)(base + L.o_vals32);
  const double* lay = (const double*)(base + L.o_layers);
  DiaDev A;
  A.d0 = v + L.ptr[0]; A.d1 = v + L.ptr[1]; A.d2 = v + L.ptr[2]; A.d3 = v + L.ptr[3];
  A.f1 = f + L.ptr[1]; A.f2 = f + L.ptr[2]; A.f3 = f + L.ptr[3];
  A.dinv = (const double*)(base + L.o_dinv);
  A.s_layer = lay + L.nz;
  A.cap_layer = lay + 2 * L.nz;
  A.n = L.n; A.nx = L.nx; A.nxny = L.nxny;
  A.ny = (int32_t)L.ny; A.nz = (int32_t)L.nz;
  A.zmarch = use_zmarch(L) ? 1 : 0; A.pad = 0;
  return A;
}

static int grid_blocks(int64_t n) {
  int64_t b = (n + (int64_t)kThreads * kRows - 1) / ((int64_t)kThreads * kRows);
  const int64_t cap = 148 * 8;           // 8 resident CTAs of 256 threads per SM, one wave
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int)b;
}

// ------------------------------------------------------------------------------------------
struct GraphEntry {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  int64_t n = 0;
  int sblocks = 0;
  int fblocks = 0;
  int device = -1;
};
static std::mutex g_mu;
static std::unordered_map<const void*, GraphEntry> g_graphs;

static cudaError_t add_kernel(cudaGraph_t g, cudaGraphNode_t* node, const cudaGraphNode_t* deps, size_t ndeps,
                              void* func, int blocks, void** args) {
  cudaKernelNodeParams kp;
  memset(&kp, 0, sizeof kp);
  kp.func = func;
  kp.gridDim = dim3((unsigned)blocks);
  kp.blockDim = dim3(kThreads);
  kp.sharedMemBytes = 0;
  kp.kernelParams = args;
  return cudaGraphAddKernelNode(node, g, deps, ndeps, &kp);
}

static int build_graph(const Workspace& w, int64_t n, int sblocks, int fblocks, GraphEntry* out) {
  const int blocks = grid_blocks(n);
  if (sblocks <= 0) sblocks = blocks;      // grid of the kernels that apply A
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
  if (fblocks > 0) {
    { void* a[] = {&ctx, &ctl, &partials};
      CU(add_kernel(body, &n_s, nullptr, 0, (void*)k_fused_pspmv, fblocks, a)); }
    { void* a[] = {&ctx, &ctl, &partials, &h_while, &h_if};
      CU(add_kernel(body, &n_u, &n_s, 1, (void*)k_update<false>, blocks, a)); }
  } else {
    { void* a[] = {&ctx, &ctl};
      CU(add_kernel(body, &n_p, nullptr, 0, (void*)k_pupdate, blocks, a)); }
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
  if (fblocks > 0) {
    void* a[] = {&ctx, &ctl};
    CU(add_kernel(ifb, &n_f, nullptr, 0, (void*)k_flush_x, blocks, a));
  }
  { void* a[] = {&ctx, &ctl, &partials, &h_while};
    CU(add_kernel(ifb, &n_t, fblocks > 0 ? &n_f : nullptr, fblocks > 0 ? 1 : 0, (void*)k_true_resid, sblocks, a)); }
  { void* a[] = {&ctx, &ctl, &partials};
    CU(add_kernel(ifb, &n_r, &n_t, 1, (void*)k_restart, blocks, a)); }

  cudaGraphExec_t ex;
  CU(cudaGraphInstantiate(&ex, g, 0));
  out->graph = g; out->exec = ex; out->n = n; out->sblocks = sblocks; out->fblocks = fblocks;
  cudaGetDevice(&out->device);
  return CUTH_OK;
}

static int get_graph(const Workspace& w, void* work_D, int64_t n, int sblocks, int fblocks, cudaGraphExec_t* ex) {
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_graphs.find(work_D);
  int dev = -1;
  cudaGetDevice(&dev);
  if (it != g_graphs.end() && (it->second.n != n || it->second.device != dev ||
                               it->second.sblocks != (sblocks > 0 ? sblocks : grid_blocks(n)) ||
                               it->second.fblocks != fblocks)) {
    cudaGraphExecDestroy(it->second.exec);
    cudaGraphDestroy(it->second.graph);
    g_graphs.erase(it);
    it = g_graphs.end();
  }
  if (it == g_graphs.end()) {
    GraphEntry e;
    int rc = build_graph(w, n, sblocks, fblocks, &e);
    if (rc != CUTH_OK) return rc;
    it = g_graphs.emplace(work_D, e).first;
  }
  *ex = it->second.exec;
  return CUTH_OK;
}

static int check_opts(const cuth_opts_t* o) {
  if (!o) return CUTH_ERR_NULL;
  if (!(o->rtol > 0.0) || o->max_iters <= 0) return CUTH_ERR_VALUE;
  if (o->precision != CUTH_FP64 && o->precision != CUTH_MIXED) return CUTH_ERR_VALUE;
  if (o->preconditioner != CUTH_PRECOND_NONE && o->preconditioner != CUTH_PRECOND_JACOBI) return CUTH_ERR_VALUE;
  return CUTH_OK;
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
  Workspace w = carve_workspace(work_D, L.n, grid->cvol_H && grid->dt > 0.0);
  DiaDev A = dev_view(dia_D, L);
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
  c.soft_restart = 1;         // promotion keeps p while the drift is small (DESIGN.md R-G11)
  c.soft_drift2 = 1e-2;       // ||t - r|| <= 0.1 ||t||
  k_set_ctx<<<1, 32, 0, st>>>(c, w.ctx, w.ctl);
  CU(cudaGetLastError());
  cudaGraphExec_t ex;
  rc = get_graph(w, work_D, L.n, stencil_blocks(L), use_zmarch(L) ? fused_blocks(L) : 0, &ex);
  if (rc) return rc;
  CU(cudaGraphLaunch(ex, st));
  return CUTH_OK;
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
  (void)opts;
  DiaLayout L;
  if (!make_layout(grid, &L)) return 0;
  return carve_workspace(nullptr, L.n, grid->cvol_H && grid->dt > 0.0).bytes;
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

int cuth_spmv(const void* dia_D, const cuth_grid_t* grid, int precision, const double* x_D, double* y_D,
              void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!dia_D || !x_D || !y_D) return CUTH_ERR_NULL;
  if (!aligned16(dia_D) || !aligned16(x_D) || !aligned16(y_D)) return CUTH_ERR_ALIGN;
  if (precision != CUTH_FP64 && precision != CUTH_MIXED) return CUTH_ERR_VALUE;
  if (x_D == y_D) return CUTH_ERR_VALUE;
  DiaDev A = dev_view(dia_D, L);
  const int sb = stencil_blocks(L);
  const int blocks = sb > 0 ? sb : grid_blocks(L.n);
  if (precision == CUTH_MIXED) k_spmv_only<true><<<blocks, kThreads, 0, (cudaStream_t)stream>>>(A, x_D, y_D);
  else k_spmv_only<false><<<blocks, kThreads, 0, (cudaStream_t)stream>>>(A, x_D, y_D);
  CU(cudaGetLastError());
  return CUTH_OK;
}

int cuth_pcg_solve(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, const double* b_D,
                   double* x_D, void* work_D, size_t work_bytes, cuth_result_t* result_D, void* stream) {
  if (!b_D) return CUTH_ERR_NULL;
  return solve_common(dia_D, grid, opts, b_D, nullptr, x_D, work_D, work_bytes, result_D, stream);
}

int cuth_transient_step(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts,
                        const double* power_D, double* T_D, void* work_D, size_t work_bytes,
                        cuth_result_t* result_D, void* stream) {
  if (!power_D) return CUTH_ERR_NULL;
  return solve_common(dia_D, grid, opts, nullptr, power_D, T_D, work_D, work_bytes, result_D, stream);
}

int cuth_profile_kernel(void* work_D, const cuth_grid_t* grid, int kernel_id, void* stream) {
  DiaLayout L;
  int rc = check_grid(grid, &L);
  if (rc) return rc;
  if (!work_D) return CUTH_ERR_NULL;
  cudaStream_t st = (cudaStream_t)stream;
  Workspace w = carve_workspace(work_D, L.n, grid->cvol_H && grid->dt > 0.0);
  const int blocks = grid_blocks(L.n);
  const int sb = stencil_blocks(L) > 0 ? stencil_blocks(L) : blocks;
  cudaGraphConditionalHandle h0 = 0;
  switch (kernel_id) {
    case -1: k_mark_no_graph<<<1, 1, 0, st>>>(w.ctl); break;
    case 0: k_pupdate<<<blocks, kThreads, 0, st>>>(w.ctx, w.ctl); break;
    case 1: k_spmv_dot<<<sb, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials); break;
    case 2: k_update<true><<<blocks, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials, h0, h0); break;
    case 4: k_fused_pspmv<<<fused_blocks(L), kThreads, 0, st>>>(w.ctx, w.ctl, w.partials); break;
    case 5: k_update<false><<<blocks, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials, h0, h0); break;
    case 3: k_true_resid<<<sb, kThreads, 0, st>>>(w.ctx, w.ctl, w.partials, h0); break;
    default: return CUTH_ERR_VALUE;
  }
  CU(cudaGetLastError());
  return CUTH_OK;
}

int cuth_set_traversal(int mode) {
  if (mode < 0 || mode > 2) return CUTH_ERR_VALUE;
  g_traversal.store(mode);
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
  return CUTH_OK;
}

const char* cuth_last_cuda_error(void) { return g_last_err.c_str(); }

int cuth_version(void) { return 10000; }

int cuth_launches_per_iteration(const cuth_grid_t* grid) {
  DiaLayout L;
  if (!make_layout(grid, &L)) return 0;
  return use_zmarch(L) ? 2 : 3;
}

}  // extern "C"
