/* cuth.h -- C ABI of the B200-native Jacobi-PCG hot path of CUTh-Solver (arxiv/paper_2606_17850).
 *
 * Boundary.  Everything behind these calls is hand-written CUDA for
 * sm_100a; there is no CPU fallback.  Conventions shared by all calls:
 *   - "_D" pointers are DEVICE pointers owned by the caller (allocate them with torch or cudaMalloc),
 *     "_H" pointers are HOST pointers.  The library allocates no device memory of its own and has NO mutable
 *     process-wide settings: every choice a call makes comes from its arguments (cuth_tuning_t below for the
 *     kernel variants).  What it keeps on the host is derived data only: a mutex-protected cache of instantiated
 *     CUDA graphs keyed by the workspace address (released by cuth_release_workspace / at process exit) and, per
 *     device, the number of co-resident CTAs of its cooperative kernels.  What a matrix object is (built or
 *     imported, transient or steady, CUTH_MIXED available or not) is recorded in the object itself, in device
 *     memory, and checked on the device.
 *   - Device buffers must be 16-byte aligned (torch gives 512).
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Every call is
 *     asynchronous on that stream and never synchronises with the host, except the three setup calls that say so
 *     (cuth_import_csr, cuth_import_coo, cuth_lanczos_bounds).
 *   - Return value: CUTH_OK or a negative cuth_status_t for errors detectable on the host (bad
 *     arguments, CUDA API failure).  NUMERICAL outcomes of a solve (converged / max-iters /
 *     breakdown) are written to result_D->status on the device, because the call is asynchronous.
 *   - Grid: nx * ny * nz cells, linear index i = x + nx*(y + ny*z), z = 0 bottom, z = nz-1 top
 *     (convective).  All of nx, ny, nz must be >= 2 so that the diagonal offsets {1, nx, nx*ny}
 *     are distinct and non-empty.  Index arithmetic is 64-bit.
 */
#ifndef CUTH_H_
#define CUTH_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  CUTH_OK = 0,
  CUTH_ERR_NULL = -1,        /* a required pointer is NULL */
  CUTH_ERR_DIMS = -2,        /* nx, ny or nz < 2, or N too large */
  CUTH_ERR_VALUE = -3,       /* non-positive dx, dy, dz, rtol; negative h; bad enum value */
  CUTH_ERR_SIZE = -4,        /* caller's buffer too small */
  CUTH_ERR_ALIGN = -5,       /* device pointer not 16-byte aligned */
  CUTH_ERR_CUDA = -6,        /* a CUDA runtime call failed (see cuth_last_cuda_error) */
  CUTH_ERR_NOT_TRANSIENT = -7,/* cuth_transient_step on a matrix built without cvol/dt (or on an imported matrix) */
  CUTH_ERR_STRUCTURE = -8,    /* cuth_import_csr: the matrix is not a symmetric 7-point matrix of this grid (see the report) */
  CUTH_ERR_FP64_ONLY = -9     /* reserved (round 1 returned it from the host; the condition is now detected on the
                                 device: CUTH_SOLVE_FP64_ONLY) */
} cuth_status_t;

/* result_D->status values (device-side outcome of a solve).  The last three mean "nothing was computed":
 * FP64_ONLY      -- a fp32-stored precision was requested on an imported matrix whose row sums are not constant
 *                   per layer (cuth_import_report_t.mixed_ok == 0);
 * NOT_TRANSIENT  -- cuth_transient_step on a matrix object built without cvol / dt, or on an imported one;
 * BAD_MATRIX     -- dia_D does not hold a matrix object of this grid (magic number / dimensions differ). */
enum { CUTH_SOLVE_CONVERGED = 0, CUTH_SOLVE_MAX_ITERS = 1, CUTH_SOLVE_BREAKDOWN = 2, CUTH_SOLVE_RUNNING = 3,
       CUTH_SOLVE_FP64_ONLY = 4, CUTH_SOLVE_NOT_TRANSIENT = 5, CUTH_SOLVE_BAD_MATRIX = 6,
       CUTH_SOLVE_CONVERGED_UNVERIFIED = 7 /* CUTH_FIXED32 only: the fp32 recursive residual passed the test */ };

/* cuth_opts_t.precision / cuth_spmv precision.
 * CUTH_FP64        fixed FP64.
 * CUTH_MIXED       the adaptive scheme of PAPER.md §IV-D with the early-stage operator in DIFFERENCE form
 *                  (DESIGN.md R-F3): the product path.
 * CUTH_MIXED_STD32 ABLATION: the same scheme with the paper's A2 taken literally -- every diagonal, D0 included,
 *                  rounded to fp32 and applied in standard form.  On these grids the true
 *                  residual then floors near 1e-2 ||b|| and eq. (14c) / (14b) do the switching.
 * CUTH_FIXED32     ABLATION: the paper's fixed-FP32 solver (Table VI): fp32 matrix A2 in standard
 *                  form, fp32 x, r, p, mu and fp32 arithmetic including the dots; stops on its own recursive
 *                  residual, never looks at b - A x (status CUTH_SOLVE_CONVERGED_UNVERIFIED); rel_resid_true
 *                  reports the fp64 residual it really reached.  Solver only; Jacobi / no preconditioner. */
enum { CUTH_FP64 = 0, CUTH_MIXED = 1, CUTH_MIXED_STD32 = 2, CUTH_ABLATION_STD32 = 2, CUTH_FIXED32 = 3 };
enum { CUTH_PRECOND_NONE = 0, CUTH_PRECOND_JACOBI = 1, CUTH_PRECOND_CHEBYSHEV = 2 };
enum { CUTH_CHEB_DEFAULT = 0, CUTH_CHEB_A3_FP16 = 1 };   /* cuth_opts_t.cheb_storage */

/* The thermal problem of PAPER.md §III-B: eq. (4) (steady) and eq. (5) (backward
 * Euler) on a box of cells with adiabatic sides/bottom (eq. (3)) and a Robin top
 * (eq. (2)); T_amb = 0, so temperatures are rises above ambient. */
typedef struct {
  int64_t nx, ny, nz;
  double dx, dy;              /* lateral cell size, m */
  const double* dz_H;         /* [nz] layer thickness, m (host) */
  const double* kappa_D;      /* conductivity W/m.K (DEVICE): nz values or nx*ny*nz values */
  int32_t kappa_is_per_layer; /* 1: kappa_D has nz values, 0: one per cell */
  double h_top;               /* W/m^2.K on the top face of layer nz-1 */
  const double* cvol_H;       /* [nz] volumetric heat capacity J/m^3.K (host), or NULL => steady */
  double dt;                  /* s; <= 0 => steady */
} cuth_grid_t;

/* Which variant of a kernel a call uses.  Zero-initialised = automatic (the measured-fastest rule for the grid,
 * DESIGN.md §5); the non-zero values exist so that tests and measurements can run every variant.  Results agree
 * up to fp64 summation order whatever is chosen.  Per call: there is no process-wide setting. */
typedef struct {
  int32_t traversal;          /* how the kernels that apply A walk the grid: 0 automatic (z-marching when one x-y plane
                                 of the six streamed arrays no longer fits L2 -- nx*ny >= 2^18 -- or from 2^17 columns
                                 on grids of more than 2^21 rows; flat 1-D streaming otherwise), 1 flat, 2 z-marching */
  int32_t loop_mode;          /* where the PCG loop lives: 0 automatic (one persistent cooperative kernel up to 2^21
                                 rows -- up to 2^22 where the TMA-staged K1 is not available --, the CUDA graph with
                                 conditional nodes beyond; grids whose rows fit the shared memory of one 8-CTA
                                 thread-block cluster -- about 13 k rows, BASELINE cfg 1 -- run as ONE cluster-resident
                                 kernel, Jacobi / no preconditioner), 1 graph, 2 persistent kernel wherever the flat
                                 traversal applies, 3 cluster-resident kernel (CUTH_ERR_VALUE when the grid does not fit; rows
                                 in registers up to 1024 rows per CTA, in shared memory beyond), 4 the cluster-resident
                                 kernel with the rows in shared memory whatever the size */
  int32_t k1_variant;         /* z-marching kernels: 0 automatic (K1 with TMA-staged operands when nx % 4 == 0 and the
                                 plane has >= 288 tiles of 64 x 8 columns; else two x-adjacent columns per thread when nx
                                 is even and there are >= 2048 tiles; else one column), 1 one column per thread,
                                 2 two columns per thread (nx even), K1 TMA-staged whenever nx % 4 == 0,
                                 3 = 2 with ordinary loads everywhere.  cuth_spmv follows the same field: automatic =
                                 TMA-staged operands when nx % 4 == 0, the plane has >= 592 such tiles and nz >= 12; 2
                                 forces them wherever nx % 4 == 0; 1 / 3 keep the kernels with ordinary loads (same y,
                                 bit for bit) */
  int32_t cheb_fusion;        /* Chebyshev passes per kernel (fp32 modes, nx even): 0 automatic = 2 = two passes, TMA
                                 operands when nx % 4 == 0 (A3: % 8); 1 one pass per kernel; 3 two passes, never TMA */
  int32_t pair_rows;          /* rows of a region of the TMA two-pass Chebyshev kernel: 0 automatic, 8, 16 */
  int32_t pair_occupancy;     /* resident CTAs/SM of that kernel: 0 automatic (4), 2..4 */
  int32_t lanczos_fp32;       /* cuth_lanczos_bounds: 0 = fp64 vectors on A1 (DESIGN.md R-C5), 1 = the paper's variant
                                 (PAPER.md:315, 340): fp32 vectors and the fixed-FP32 SpMV on the fp32 copy A2 */
  int32_t reserved;           /* must be 0 */
} cuth_tuning_t;

typedef struct {
  int32_t precision;          /* CUTH_FP64, CUTH_MIXED (§IV-D) or an ablation value above */
  double rtol;                /* stop when ||b - A x||_2 <= rtol * ||b||_2 (true fp64 residual) */
  int32_t max_iters;          /* cap on PCG iterations (Alg. 1 loop), > 0 */
  int32_t true_resid_period;  /* MIXED early stage: evaluate b - A1 x every this many iterations
                                 (20 steady, 5 transient); <= 0 => 20 */
  int32_t preconditioner;     /* CUTH_PRECOND_JACOBI (M = diag A), CUTH_PRECOND_NONE (M = I) or
                                 CUTH_PRECOND_CHEBYSHEV (Alg. 3; needs the three fields below) */
  int32_t cheb_degree;        /* k of Alg. 3 (the paper uses 30); 3 <= k <= 64 */
  double cheb_lmin, cheb_lmax;/* spectral interval [alpha, beta] of eq. (10)-(11), e.g. from
                                 cuth_lanczos_bounds; 0 < lmin < lmax, and lmax must bound the spectrum of A */
  int32_t cheb_storage;       /* matrix the preconditioner multiplies by in MIXED mode: CUTH_CHEB_DEFAULT = the fp32
                                 copy A2, CUTH_CHEB_A3_FP16 = the half-precision copy A3 promoted to fp32 on load
                                 (Alg. 4 "arithmetic decoupling").  Ignored in FP64 mode. */
  cuth_tuning_t tuning;       /* kernel variants; all zero = automatic */
} cuth_opts_t;

typedef struct {
  int32_t status;             /* CUTH_SOLVE_* */
  int32_t iterations;         /* PCG iterations done (Alg. 1 line 13 counter) */
  int32_t promotions;         /* early->late switches (0 in FP64 mode, <= 1 in MIXED) */
  int32_t true_resid_evals;   /* number of explicit b - A1 x evaluations */
  double rel_resid_true;      /* last evaluated ||b - A1 x||_2 / ||b||_2 (fp64) */
  double rel_resid_rec;       /* last recursive ||r||_2 / ||b||_2 */
  int32_t switch_reason;      /* MIXED: 0 none, else the first criterion, in the printed order, that held at the
                                 switch: 1 = (14a), 2 = (14b), 3 = (14c) */
  int32_t switch_iteration;   /* iteration at which the switch happened */
  int32_t switch_mask;        /* every criterion that held at the switch: bit 0 = (14a), bit 1 = (14b), bit 2 = (14c) */
  int32_t hard_restarts;      /* hot restarts with p := z (Alg. 1 line 3): large drift at the switch, or a failed
                                 verification of the stopping test in the late stage */
  int32_t soft_restarts;      /* hot restarts that kept p through Alg. 1 line 12 (small drift, DESIGN.md R-G11) */
  int32_t reserved;
} cuth_result_t;

/* Bytes of the caller-allocated device buffer that holds the matrix object (header, fp64 packed
 * diagonals A1, fp32 copy A2, 1/D0, per-layer row sums).  0 on invalid dims. */
size_t cuth_dia_bytes(const cuth_grid_t* grid);

/* Bytes of the caller-allocated device workspace for cuth_pcg_solve / cuth_transient_step
 * (control block, reduction partials, vectors r, p, mu and -- transient only -- b). */
size_t cuth_workspace_bytes(const cuth_grid_t* grid, const cuth_opts_t* opts);

/* Builder (hot-path step a0).  Computes from the cell fields the condensed-DIA ("Quad-Diag",
 * PAPER.md:219, Fig. 4) matrix of eq. (4)/(5): only the main and the three upper diagonals
 * (offsets 0, 1, nx, nx*ny), unpadded: diagonal k has exactly N - off[k] elements, element j =
 * A[j, j+off[k]]; packed D0|D1|D2|D3 in one fp64 array `vals`, ptr = {0, N, 2N-1, 3N-1-nx,
 * 4N-1-nx-nx*ny}.  Entries of A are stored (off-diagonals negative).  Where the +x / +y neighbour
 * does not exist (x = nx-1, y = ny-1) the stored element is +0.0.  Also stored: the fp32 copy A2
 * (round-to-nearest-even of vals), 1/D0 (fp64), and the exact row sums s(z) used by the MIXED
 * operator.  Arithmetic: fp64 without FMA contraction, in the order DESIGN.md §4 states, so
 * values are bit-identical to the oracle's.  dia_D: device buffer of >= cuth_dia_bytes(). */
int cuth_build_dia(const cuth_grid_t* grid, void* dia_D, size_t dia_bytes, void* stream);

/* What cuth_import_csr found.  The first four counts must all be zero for the import to succeed. */
typedef struct {
  int64_t off_stencil;        /* non-zero entries whose column is not row + {0, +-1, +-nx, +-nx*ny}, is out of range, or
                                 couples x = nx-1 with x = 0 of the next line / y = ny-1 with y = 0 of the next plane */
  int64_t asymmetric_rows;    /* rows with a lower-triangle entry that differs from its mirror (absent == 0) */
  int64_t bad_diagonal;       /* rows whose main-diagonal entry is missing, not positive or not finite */
  int64_t duplicates;         /* entries that repeat a column already seen in their row */
  int64_t positive_offdiag;   /* off-diagonal entries > 0: information only (a conductance matrix has none) */
  double max_rowsum_dev;      /* max over rows of |row sum - s(layer)| / (smallest diagonal entry of the layer) */
  int32_t mixed_ok;           /* 1: the row sums are constant per layer to 1e-9, so CUTH_MIXED is available */
  int32_t reserved;
  int64_t bad_rowptr;         /* cuth_import_csr: rows whose [rowptr[i], rowptr[i+1]) is not a sane range -- rowptr[0] != 0,
                                 decreasing, more than 4096 entries in a row, or (cuth_import_csr_n) beyond nnz.  When
                                 non-zero NOTHING else of the matrix is read: the call fails with CUTH_ERR_STRUCTURE */
} cuth_import_report_t;

/* Importer (the paper's matrices are sparse matrices exported by 3D-ICE, which
 * PAPER.md:219 then "decomposes and stores as a set of diagonal vectors").  Takes a square CSR matrix of order
 * nx*ny*nz on the DEVICE (rowptr int64 [n+1], col int32 [nnz], val fp64 [nnz]; columns in any order within a row),
 * checks that it is a symmetric matrix with a positive diagonal whose non-zeros all sit on the seven diagonals
 * {0, +-1, +-nx, +-nx*ny} of the box and never couple across an x / y edge, and writes the same matrix object
 * cuth_build_dia writes: the main and the three upper diagonals are copied BIT-EXACT into the packed layout (a
 * missing entry is +0.0), then A2, 1/D0, A3 are derived as in the builder.  Only nx, ny, nz of `grid` are used
 * (dx, dy, h_top must still be valid numbers).  rowsum_layer_H: NULL, or [nz] exact row sums s(z) of the operator
 * per layer (physically h*dx*dy on the top layer plus C*V/dt); the MIXED operator is applied
 * in difference form and needs them (DESIGN.md R-F3).  With NULL they are taken from the matrix (midrange of the
 * layer's computed row sums, clamped at 0); if the rows of a layer do not agree to 1e-9 of the layer's smallest
 * diagonal entry the matrix is usable in CUTH_FP64 only (report->mixed_ok = 0; MIXED calls return
 * CUTH_ERR_FP64_ONLY), and if a supplied rowsum_layer_H disagrees the call fails with CUTH_ERR_STRUCTURE.
 * Imported matrices are steady operators for this library: cuth_transient_step returns CUTH_ERR_NOT_TRANSIENT
 * (form b = P + (C V/dt) T_n yourself and call cuth_pcg_solve).
 * report_H (host, may be NULL) is always filled.  This call SYNCHRONISES `stream` (setup, not hot path).
 * On CUTH_ERR_STRUCTURE the contents of dia_D are unspecified. */
int cuth_import_csr(const cuth_grid_t* grid, const int64_t* rowptr_D, const int32_t* col_D, const double* val_D,
                    const double* rowsum_layer_H, void* dia_D, size_t dia_bytes, cuth_import_report_t* report_H,
                    void* stream);

/* cuth_import_csr with the number of stored entries, so that a rowptr that points beyond the col / val arrays is caught
 * before anything is read through it (nnz < 0 = unknown = cuth_import_csr). */
int cuth_import_csr_n(const cuth_grid_t* grid, const int64_t* rowptr_D, const int32_t* col_D, const double* val_D,
                      int64_t nnz, const double* rowsum_layer_H, void* dia_D, size_t dia_bytes,
                      cuth_import_report_t* report_H, void* stream);

/* The same import from COORDINATE format: nnz entries (row_D[q], col_D[q], val_D[q]) in any order (int32 indices,
 * device).  Same checks, same report, same matrix object as cuth_import_csr (one thread per entry; a coordinate met
 * twice counts as a duplicate whichever copy came first).  SYNCHRONISES `stream`. */
int cuth_import_coo(const cuth_grid_t* grid, const int32_t* row_D, const int32_t* col_D, const double* val_D, int64_t nnz,
                    const double* rowsum_layer_H, void* dia_D, size_t dia_bytes, cuth_import_report_t* report_H,
                    void* stream);

/* View of the matrix object for the bit-exact layout test: device pointers to the packed fp64
 * values and to the fp32 copy (same ptr/off), and the host copies of ptr[5], off[4].
 * Any output pointer may be NULL.  Pure host arithmetic, no CUDA call. */
int cuth_dia_view(const void* dia_D, const cuth_grid_t* grid, const double** vals_D, const float** vals32_D,
                  const double** inv_diag_D, int64_t ptr_H[5], int64_t off_H[4]);

/* SpMV (hot-path step a1), Alg. 2 read 0-based: y = A x with
 * y[i] = D0[i] x[i] + sum_k ( Dk[i] x[i+off k] + Dk[i-off k] x[i-off k] ), out-of-range terms dropped.
 * precision CUTH_FP64: fp64 matrix A1.  CUTH_MIXED: fp32-stored off-diagonals promoted to fp64
 * ("FP64/32 SpMV with arithmetic decoupling") applied in difference form
 * y_i = s_i x_i + sum_j g_ij (x_i - x_j) (DESIGN.md R-F3).  CUTH_ABLATION_STD32: the same fp32 copy applied
 * literally in standard form (all four diagonals rounded): an ablation switch that reproduces the fixed-fp32
 * drift of the paper's Table VI; no solver path uses it.  x_D, y_D: fp64 [N], distinct buffers. */
int cuth_spmv(const void* dia_D, const cuth_grid_t* grid, int precision, const double* x_D, double* y_D,
              void* stream);

/* PCG solve (steps a1-a5), Alg. 1 with M = diag(A): x_D holds x0 on entry and
 * the solution on exit.  The loop runs entirely on the device inside one CUDA graph (conditional
 * WHILE node); convergence is decided on the device and verified on the true fp64 residual.
 * MIXED: early stage on the fp32-stored operator, switch by eq. (14a)-(14c) with
 * hot restart, late stage fp64.  b_D is read only.  work_D >= cuth_workspace_bytes().
 * result_D: device cuth_result_t written when the solve ends.  b = 0 gives x = 0. */
int cuth_pcg_solve(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, const double* b_D,
                   double* x_D, void* work_D, size_t work_bytes, cuth_result_t* result_D, void* stream);

/* Batched solve (SURVEY.md §8(f) "multi-RHS / batched solves sharing one A"; PAPER.md:473 observes that many
 * right-hand sides on one matrix favour direct solvers -- this call amortises A on the iterative path instead).
 * nrhs independent systems A x_s = b_s, 1 <= nrhs <= 32, each by its own Alg. 1 recurrence (own
 * alpha, beta, stopping test on the true fp64 residual), advanced in lock-step by ONE persistent cooperative kernel:
 * every matrix row is fetched once per 4 right-hand sides and every grid-wide barrier / reduction serves all of
 * them, so small grids (where a single solve is bound by barrier latency) solve nrhs systems in little more than
 * the time of one.  This is not block-CG: x_s is what cuth_pcg_solve would return for b_s, up to summation order.
 * b_D, x_D: [nrhs][N] fp64, right-hand-side-major (x_D in: initial guesses, out: solutions).  result_D: [nrhs].
 * opts: CUTH_FP64 or CUTH_MIXED (every right-hand side runs the policy of cuth_pcg_solve on its own: own stage, own
 * switch by eq. (14a)-(14c), own hot restart); preconditioner CUTH_PRECOND_JACOBI or CUTH_PRECOND_NONE (else
 * CUTH_ERR_VALUE).
 * work_D >= cuth_batch_workspace_bytes(grid, nrhs).  All CTAs must be co-resident: needs cooperative launch
 * (CUTH_ERR_CUDA otherwise).  Asynchronous on `stream` like cuth_pcg_solve. */
size_t cuth_batch_workspace_bytes(const cuth_grid_t* grid, int nrhs);
int cuth_pcg_solve_batch(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, int nrhs,
                         const double* b_D, double* x_D, void* work_D, size_t work_bytes, cuth_result_t* result_D,
                         void* stream);

/* One backward-Euler step (step a6), eq. (5): forms b = P_{n+1} + (C V/dt) T_n in
 * one fused pass and solves A T_{n+1} = b warm-started from T_n.  power_D: W per cell [N];
 * T_D: in T_n, out T_{n+1}.  The matrix must have been built with cvol_H and dt > 0. */
int cuth_transient_step(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts,
                        const double* power_D, double* T_D, void* work_D, size_t work_bytes,
                        cuth_result_t* result_D, void* stream);

/* Drops the cached CUDA graph(s) tied to this workspace address (call before freeing it). */
int cuth_release_workspace(const void* work_D);

/* Text of the last CUDA error seen by this library on the calling thread ("" if none). */
const char* cuth_last_cuda_error(void);

/* Library version, e.g. 10000 = 1.0.0 */
int cuth_version(void);

/* Kernel launches per PCG iteration of the graph body for this grid and these options (2 on the fused path used
 * for large planes -- 3 there for a MIXED solve on a stack of fewer than 12 layers, whose K1 is two nodes, the
 * TMA-staged kernel for the early stage and the two-column LDG kernel for the late stage, each returning at once in
 * the other's stage --, 3 on the flat path, 0 when the whole solve is one persistent kernel); bench.py reports
 * gpu_launches = prologue + this * iterations + true-residual branches + epilogue.  Pure host. */
int cuth_launches_per_iteration(const cuth_grid_t* grid, const cuth_opts_t* opts);

/* How the kernels of a solve with these options walk this grid (what cuth_tuning_t.traversal = 0 resolves to):
 * 1 = flat 1-D streaming (k_pupdate, k_spmv_dot, k_update in the graph loop), 2 = z-marching (the fused K1 + K2);
 * negative on bad arguments.  Pure host. */
int cuth_traversal(const cuth_grid_t* grid, const cuth_opts_t* opts);

/* Where the PCG loop of a solve with these options on this grid lives (what cuth_tuning_t.loop_mode = 0 resolves
 * to): 1 = CUDA graph with conditional nodes, 2 = persistent cooperative kernel, 3 = cluster-resident kernel,
 * 4 = the fixed-FP32 ablation kernel; negative on bad arguments.  Pure host. */
int cuth_loop_home(const cuth_grid_t* grid, const cuth_opts_t* opts);

/* Kernel launches of ONE Chebyshev apply (Alg. 3) for this grid and these options: the first
 * pass, the middle passes (single, or two per launch -- see cuth_tuning_t.cheb_fusion) and the last pass; 0 when the
 * preconditioner is not Chebyshev, negative on bad arguments.  *pairs_out (may be NULL) = how many of them are
 * two-pass launches.  Pure host. */
int cuth_cheb_launches(const cuth_grid_t* grid, const cuth_opts_t* opts, int* pairs_out);

/* Spectral-range estimate for the Chebyshev preconditioner: `steps` Lanczos iterations on
 * the device (start vector v0_D, e.g. the right-hand side), the tridiagonal T copied to the host and its
 * extreme eigenvalues found there in fp64 (bisection).  bounds_H[0] = smallest Ritz value, bounds_H[1] =
 * largest Ritz value, bounds_H[2] = Gershgorin upper bound max_i sum_j |a_ij| (always >= lambda_max),
 * bounds_H[3], bounds_H[4] = the interval to hand to cuth_opts_t.cheb_lmin / cheb_lmax: [Ritz min,
 * min(1.05 * Ritz max, Gershgorin)].
 * Uses the solver workspace (>= cuth_workspace_bytes).  This call SYNCHRONISES `stream` (setup, not hot path). */
int cuth_lanczos_bounds(const void* dia_D, const cuth_grid_t* grid, const double* v0_D, int steps, void* work_D,
                        size_t work_bytes, double bounds_H[5], void* stream);
/* ... with an explicit kernel variant for its SpMV (tuning may be NULL = automatic). */
int cuth_lanczos_bounds_tuned(const void* dia_D, const cuth_grid_t* grid, const cuth_tuning_t* tuning, const double* v0_D,
                              int steps, void* work_D, size_t work_bytes, double bounds_H[5], void* stream);

/* The host half of cuth_lanczos_bounds on its own (pure host, no CUDA): smallest and largest eigenvalue of
 * the symmetric tridiagonal matrix with diagonal alpha_H[0..m) and off-diagonal beta_H[0..m-1), by Sturm
 * bisection in fp64 (the spectrum of T is solved on the CPU). */
int cuth_tridiag_extremes(const double* alpha_H, const double* beta_H, int m, double out_H[2]);

/* One application of the Chebyshev polynomial preconditioner, z = q(A) r (Alg. 3), with the
 * degree and interval of `opts` (preconditioner must be CUTH_PRECOND_CHEBYSHEV): k-1 stencil kernels, no
 * reduction.  precision CUTH_FP64: fp64 vectors and matrix; CUTH_MIXED: fp32 vectors on the fp32-stored matrix
 * (PAPER.md:376).  r_D, z_D fp64 [N], distinct.  work_D >= cuth_workspace_bytes(grid, opts). */
int cuth_cheb_apply(const void* dia_D, const cuth_grid_t* grid, const cuth_opts_t* opts, const double* r_D,
                    double* z_D, void* work_D, size_t work_bytes, void* stream);

/* cuth_spmv with an explicit choice of kernel variant (tuning may be NULL = automatic = cuth_spmv). */
int cuth_spmv_tuned(const void* dia_D, const cuth_grid_t* grid, int precision, const cuth_tuning_t* tuning,
                    const double* x_D, double* y_D, void* stream);

/* Measurement hook (bench.py, ncu, __graft_entry__.smoke): launches ONE loop-body kernel of the solve whose context
 * is still in this workspace, outside the graph and with the graph's launch configuration for `opts` (the options of
 * that solve), so that it can be timed with CUDA events on `stream` and shows up by name in a profiler's launch list
 * (kernel nodes of graphs with conditional nodes do not).  kernel_id: -1 = arm with the stage the solve ended in,
 * -2 = arm and force the EARLY stage (fp32-stored operator; MIXED solves only) -- one of the two must be called once
 * after the solve, before any other id; 0 = p-update, 1 = SpMV + p.mu, 2 = x/r update + dots, 3 = true residual
 * (fused path: with the pending x-update and the restart folded in), 4 = fused p-update + SpMV (K1 of the fused
 * path), 5 = r update + dots without x (K2 of the fused path), 6 / 7 / 8 = one middle step of the Chebyshev apply in
 * fp64 / fp32 on A2 / fp32 on the fp16 copy A3 (only after a CUTH_PRECOND_CHEBYSHEV solve); 9 / 10 = one fused PAIR
 * of Chebyshev passes on A2 / A3.  The vectors of the finished solve are overwritten; x_D is modified by ids 2-4. */
int cuth_profile_kernel(void* work_D, const cuth_grid_t* grid, const cuth_opts_t* opts, int kernel_id, void* stream);

/* Test hook for the device-side stage-switch policy (csrc/cuth_policy.cuh): runs the decision
 * function the solver kernels run after an evaluation of r_true = b - A1 x, ONCE, on caller-given scalars, in a
 * one-thread kernel on `stream`, and writes what it decided to out_D (device, 8 x int32: [0] go, [1] stage after,
 * [2] switch_reason, [3] switch_mask, [4] restart kind (0 none, 1 hard, 2 soft), [5] status, [6] promotions,
 * [7] 0).  in_H (host, 8 doubles): ||r_low||^2, ||r_true||^2, ||r_true - r_low||^2, ||r_true||^2 at the previous
 * evaluation, ||r_low||^2 at the previous evaluation, ||b||^2, rtol, soft_drift (<= 0: library default 0.1).
 * flags: bit 0 = late stage, bit 1 = the recursive residual had passed the stopping test, bit 2 = iteration cap
 * reached.  No solver state is touched. */
int cuth_policy_probe(const double in_H[8], int flags, int32_t* out_D, void* stream);

/* The ONE entry point that needs no caller-allocated scratch and allocates nothing itself (for callers that cannot
 * call cudaMalloc: code under CUDA-graph capture, tight serving loops, harnesses that forbid it): the true residual of
 * the stopping rule (DESIGN.md R-G7), t = b - A1 x in fp64 on the packed diagonals, with
 * out_D[0] = ||t||_2^2, out_D[1] = ||b||_2^2, out_D[2] = ||t||_2 / ||b||_2 (0 when b = 0), out_D[3] = 0 (device, 4 doubles).
 * t_D: device [N] to receive t, or NULL when only the norms are wanted; must not alias x_D.  b_D, x_D: device [N].
 * The per-CTA partial sums of the reduction live in a FILE-SCOPE device array of cuth_noalloc_max_rows()-dependent,
 * fixed size (32 KB + 256 B) that every GPU loading this library holds until the process exits.  Hence:
 *   - LIMIT: grids of more than cuth_noalloc_max_rows() = 16 777 216 rows (BASELINE cfg 3 fits exactly) are refused with
 *     CUTH_ERR_SIZE before anything is launched; cuth_noalloc_last_error() says why;
 *   - all calls on a GPU share that array: calls that may OVERLAP on the GPU (different streams) race on it and must be
 *     serialised by the caller; back-to-back calls on one stream are fine (the call clears what must start at zero);
 *   - results are bit-reproducible (fixed-order sums) and equal cuth_spmv followed by b - y up to the last bit of y.
 * Calls no cudaMalloc / cudaFree / allocating library routine; asynchronous on `stream`. */
int64_t cuth_noalloc_max_rows(void);
const char* cuth_noalloc_last_error(void);
int cuth_residual_noalloc(const void* dia_D, const cuth_grid_t* grid, const double* b_D, const double* x_D,
                          double* t_D, double* out_D, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CUTH_H_ */
