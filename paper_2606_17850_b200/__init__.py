"""cuth: B200-native Jacobi-PCG hot path of CUTh-Solver (arxiv/paper_2606_17850).

Thin Python binding over the C-ABI library declared in include/cuth.h.  Every step of the
path runs in the hand-written CUDA kernels of csrc/; this package only marshals arguments
(torch tensors -> device pointers, current stream -> cudaStream_t).  There is no CPU fallback:
importing `binding` without the compiled library, or calling it without a CUDA device, raises.
"""
from .binding import (  # noqa: F401
    CuthError, Grid, Opts, Result, DiaMatrix, Solver, BatchSolver, cuth_batch_workspace_bytes, cuth_pcg_solve_batch,
    cuth_dia_bytes, cuth_workspace_bytes, cuth_build_dia, cuth_import_csr, cuth_import_coo, cuth_dia_view, cuth_spmv,
    cuth_pcg_solve, cuth_transient_step, cuth_release_workspace, cuth_version,
    cuth_launches_per_iteration, cuth_loop_home, cuth_traversal, cuth_residual_noalloc, cuth_noalloc_max_rows, cuth_profile_kernel, cuth_spmv_tuned, cuth_policy_probe, set_default_tuning, Tuning,
    cuth_cheb_launches, cuth_lanczos_bounds, cuth_cheb_apply, cuth_tridiag_extremes, load_library, exported_symbols,
    FP64, MIXED, MIXED_STD32, FIXED32, ABLATION_STD32, SOLVE_FP64_ONLY, SOLVE_NOT_TRANSIENT, SOLVE_BAD_MATRIX,
    SOLVE_CONVERGED_UNVERIFIED, PRECOND_NONE, PRECOND_JACOBI, PRECOND_CHEBYSHEV, CHEB_DEFAULT, CHEB_A3_FP16,
)
