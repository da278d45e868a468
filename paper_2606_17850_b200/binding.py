"""ctypes binding with the same names as include/cuth.h (argument marshalling only)."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("CUTH_LIB", os.path.join(HERE, "libcuth.so"))   # CUTH_LIB: developer override

FP64, MIXED, MIXED_STD32, FIXED32 = 0, 1, 2, 3
ABLATION_STD32 = MIXED_STD32
PRECOND_NONE, PRECOND_JACOBI, PRECOND_CHEBYSHEV = 0, 1, 2
CHEB_DEFAULT, CHEB_A3_FP16 = 0, 1
STATUS_NAMES = {0: "converged", 1: "max_iters", 2: "breakdown", 3: "running", 4: "fp64_only", 5: "not_transient",
                6: "bad_matrix", 7: "converged_unverified"}
SOLVE_FP64_ONLY, SOLVE_NOT_TRANSIENT, SOLVE_BAD_MATRIX, SOLVE_CONVERGED_UNVERIFIED = 4, 5, 6, 7
_ERR = {-1: "CUTH_ERR_NULL", -2: "CUTH_ERR_DIMS", -3: "CUTH_ERR_VALUE", -4: "CUTH_ERR_SIZE",
        -5: "CUTH_ERR_ALIGN", -6: "CUTH_ERR_CUDA", -7: "CUTH_ERR_NOT_TRANSIENT", -8: "CUTH_ERR_STRUCTURE",
        -9: "CUTH_ERR_FP64_ONLY"}


class CuthError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = _ERR.get(code, str(code))
        if code == -6:
            msg += ": " + load_library().cuth_last_cuda_error().decode()
        super().__init__(f"{where} failed: {msg}")


class cuth_grid_t(C.Structure):
    _fields_ = [("nx", C.c_int64), ("ny", C.c_int64), ("nz", C.c_int64),
                ("dx", C.c_double), ("dy", C.c_double),
                ("dz_H", C.c_void_p), ("kappa_D", C.c_void_p), ("kappa_is_per_layer", C.c_int32),
                ("h_top", C.c_double), ("cvol_H", C.c_void_p), ("dt", C.c_double)]


class cuth_tuning_t(C.Structure):
    _fields_ = [("traversal", C.c_int32), ("loop_mode", C.c_int32), ("k1_variant", C.c_int32),
                ("cheb_fusion", C.c_int32), ("pair_rows", C.c_int32), ("pair_occupancy", C.c_int32),
                ("lanczos_fp32", C.c_int32), ("reserved", C.c_int32)]


class cuth_opts_t(C.Structure):
    _fields_ = [("precision", C.c_int32), ("rtol", C.c_double), ("max_iters", C.c_int32),
                ("true_resid_period", C.c_int32), ("preconditioner", C.c_int32),
                ("cheb_degree", C.c_int32), ("cheb_lmin", C.c_double), ("cheb_lmax", C.c_double),
                ("cheb_storage", C.c_int32), ("tuning", cuth_tuning_t)]


class cuth_result_t(C.Structure):
    _fields_ = [("status", C.c_int32), ("iterations", C.c_int32), ("promotions", C.c_int32),
                ("true_resid_evals", C.c_int32), ("rel_resid_true", C.c_double),
                ("rel_resid_rec", C.c_double), ("switch_reason", C.c_int32),
                ("switch_iteration", C.c_int32), ("switch_mask", C.c_int32), ("hard_restarts", C.c_int32),
                ("soft_restarts", C.c_int32), ("reserved", C.c_int32)]


class cuth_import_report_t(C.Structure):
    _fields_ = [("off_stencil", C.c_int64), ("asymmetric_rows", C.c_int64), ("bad_diagonal", C.c_int64),
                ("duplicates", C.c_int64), ("positive_offdiag", C.c_int64), ("max_rowsum_dev", C.c_double),
                ("mixed_ok", C.c_int32), ("reserved", C.c_int32), ("bad_rowptr", C.c_int64)]


EXPORTS = ["cuth_import_csr", "cuth_import_coo", "cuth_batch_workspace_bytes", "cuth_pcg_solve_batch", "cuth_dia_bytes",
           "cuth_workspace_bytes", "cuth_build_dia", "cuth_dia_view", "cuth_spmv", "cuth_spmv_tuned", "cuth_pcg_solve",
           "cuth_transient_step", "cuth_release_workspace", "cuth_last_cuda_error", "cuth_version",
           "cuth_launches_per_iteration", "cuth_profile_kernel", "cuth_lanczos_bounds", "cuth_lanczos_bounds_tuned",
           "cuth_cheb_apply", "cuth_tridiag_extremes", "cuth_cheb_launches", "cuth_policy_probe", "cuth_loop_home", "cuth_traversal",
           "cuth_residual_noalloc", "cuth_noalloc_max_rows", "cuth_noalloc_last_error", "cuth_import_csr_n"]

_lib = None


def exported_symbols():
    return list(EXPORTS)


def load_library():
    """dlopen the in-tree libcuth.so; fails loudly when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_17850_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, gp, op = C.c_void_p, C.POINTER(cuth_grid_t), C.POINTER(cuth_opts_t)
    L.cuth_dia_bytes.restype = C.c_size_t
    L.cuth_dia_bytes.argtypes = [gp]
    L.cuth_workspace_bytes.restype = C.c_size_t
    L.cuth_workspace_bytes.argtypes = [gp, op]
    L.cuth_build_dia.restype = C.c_int
    L.cuth_build_dia.argtypes = [gp, vp, C.c_size_t, vp]
    L.cuth_import_csr.restype = C.c_int
    L.cuth_import_csr.argtypes = [gp, vp, vp, vp, vp, vp, C.c_size_t, C.POINTER(cuth_import_report_t), vp]
    L.cuth_import_coo.restype = C.c_int
    L.cuth_import_coo.argtypes = [gp, vp, vp, vp, C.c_int64, vp, vp, C.c_size_t, C.POINTER(cuth_import_report_t), vp]
    L.cuth_dia_view.restype = C.c_int
    L.cuth_dia_view.argtypes = [vp, gp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp),
                                C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.cuth_spmv.restype = C.c_int
    L.cuth_spmv.argtypes = [vp, gp, C.c_int, vp, vp, vp]
    L.cuth_spmv_tuned.restype = C.c_int
    L.cuth_spmv_tuned.argtypes = [vp, gp, C.c_int, C.POINTER(cuth_tuning_t), vp, vp, vp]
    L.cuth_pcg_solve.restype = C.c_int
    L.cuth_pcg_solve.argtypes = [vp, gp, op, vp, vp, vp, C.c_size_t, vp, vp]
    L.cuth_batch_workspace_bytes.restype = C.c_size_t
    L.cuth_batch_workspace_bytes.argtypes = [gp, C.c_int]
    L.cuth_pcg_solve_batch.restype = C.c_int
    L.cuth_pcg_solve_batch.argtypes = [vp, gp, op, C.c_int, vp, vp, vp, C.c_size_t, vp, vp]
    L.cuth_transient_step.restype = C.c_int
    L.cuth_transient_step.argtypes = [vp, gp, op, vp, vp, vp, C.c_size_t, vp, vp]
    L.cuth_release_workspace.restype = C.c_int
    L.cuth_release_workspace.argtypes = [vp]
    L.cuth_last_cuda_error.restype = C.c_char_p
    L.cuth_version.restype = C.c_int
    L.cuth_launches_per_iteration.restype = C.c_int
    L.cuth_launches_per_iteration.argtypes = [gp, op]
    L.cuth_lanczos_bounds.restype = C.c_int
    L.cuth_lanczos_bounds.argtypes = [vp, gp, vp, C.c_int, vp, C.c_size_t, C.POINTER(C.c_double), vp]
    L.cuth_lanczos_bounds_tuned.restype = C.c_int
    L.cuth_lanczos_bounds_tuned.argtypes = [vp, gp, C.POINTER(cuth_tuning_t), vp, C.c_int, vp, C.c_size_t,
                                            C.POINTER(C.c_double), vp]
    L.cuth_policy_probe.restype = C.c_int
    L.cuth_policy_probe.argtypes = [C.POINTER(C.c_double), C.c_int, vp, vp]
    L.cuth_cheb_apply.restype = C.c_int
    L.cuth_cheb_apply.argtypes = [vp, gp, op, vp, vp, vp, C.c_size_t, vp]
    L.cuth_profile_kernel.restype = C.c_int
    L.cuth_profile_kernel.argtypes = [vp, gp, op, C.c_int, vp]
    _lib = L
    return L


def _check(rc, where):
    if rc != 0:
        raise CuthError(rc, where)


# ------------------------------------------------------------------ argument holders
class Grid:
    """Holds a cuth_grid_t and keeps the host arrays / device tensor it points to alive."""

    def __init__(self, nx, ny, nz, dx, dy, dz, kappa, h_top, cvol=None, dt=0.0):
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.n = self.nx * self.ny * self.nz
        self._dz = np.ascontiguousarray(dz, dtype=np.float64)
        self._cvol = None if cvol is None else np.ascontiguousarray(cvol, dtype=np.float64)
        self.kappa = kappa          # torch CUDA float64 tensor (nz or n values) or None
        per_layer = 1
        kptr = None
        if kappa is not None:
            per_layer = 1 if kappa.numel() == self.nz else 0
            kptr = kappa.data_ptr()
        self.c = cuth_grid_t(self.nx, self.ny, self.nz, float(dx), float(dy),
                             self._dz.ctypes.data, kptr, per_layer, float(h_top),
                             None if self._cvol is None else self._cvol.ctypes.data, float(dt))

    @property
    def transient(self):
        return self._cvol is not None and self.c.dt > 0

    def ref(self):
        return C.byref(self.c)


# The C library has no process-wide settings (include/cuth.h); the kernel variants travel in every call's
# cuth_tuning_t.  For the test suite and bench.py, which run whole groups of calls under one variant, THIS PYTHON
# MODULE keeps a default tuning that Opts() / DiaMatrix.spmv / the hooks below copy into their arguments.
_DEFAULT_TUNING = dict(traversal=0, loop_mode=0, k1_variant=0, cheb_fusion=0, pair_rows=0, pair_occupancy=0,
                       lanczos_fp32=0)


def set_default_tuning(**kw):
    """Python-side default for the `tuning` argument of the calls made through this binding (0 = automatic)."""
    for k, v in kw.items():
        if k not in _DEFAULT_TUNING:
            raise KeyError(k)
        _DEFAULT_TUNING[k] = int(v)


def Tuning(**kw):
    d = dict(_DEFAULT_TUNING)
    d.update({k: int(v) for k, v in kw.items()})
    return cuth_tuning_t(d["traversal"], d["loop_mode"], d["k1_variant"], d["cheb_fusion"], d["pair_rows"],
                         d["pair_occupancy"], d["lanczos_fp32"], 0)


def Opts(precision=FP64, rtol=1e-8, max_iters=200000, true_resid_period=20, preconditioner=PRECOND_JACOBI,
         cheb_degree=30, cheb_lmin=0.0, cheb_lmax=0.0, cheb_storage=CHEB_DEFAULT, tuning=None):
    return cuth_opts_t(int(precision), float(rtol), int(max_iters), int(true_resid_period), int(preconditioner),
                       int(cheb_degree), float(cheb_lmin), float(cheb_lmax), int(cheb_storage),
                       tuning if tuning is not None else Tuning())


@dataclass
class Result:
    status: int
    iterations: int
    promotions: int
    true_resid_evals: int
    rel_resid_true: float
    rel_resid_rec: float
    switch_reason: int
    switch_iteration: int
    switch_mask: int = 0
    hard_restarts: int = 0
    soft_restarts: int = 0

    @property
    def status_name(self):
        return STATUS_NAMES.get(self.status, "?")


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


# ------------------------------------------------------------------ the C calls, same names
def cuth_dia_bytes(grid: Grid) -> int:
    return int(load_library().cuth_dia_bytes(grid.ref()))


def cuth_workspace_bytes(grid: Grid, opts) -> int:
    return int(load_library().cuth_workspace_bytes(grid.ref(), C.byref(opts)))


def cuth_build_dia(grid: Grid, dia, stream=None):
    _check(load_library().cuth_build_dia(grid.ref(), _ptr(dia), dia.numel() * dia.element_size(),
                                         stream or _stream()), "cuth_build_dia")


def cuth_import_csr(grid: Grid, rowptr, col, val, dia, rowsum_layer=None, stream=None, check=True, nnz=None):
    """rowptr int64 / col int32 / val float64 CUDA tensors.  Returns the cuth_import_report_t; raises CuthError on
    failure unless check=False (then returns (rc, report)).  Synchronises the stream."""
    import torch
    assert rowptr.dtype == torch.int64 and col.dtype == torch.int32 and val.dtype == torch.float64
    rep = cuth_import_report_t()
    rs = None if rowsum_layer is None else np.ascontiguousarray(rowsum_layer, dtype=np.float64)
    L = load_library()
    L.cuth_import_csr_n.restype = C.c_int
    L.cuth_import_csr_n.argtypes = [C.POINTER(cuth_grid_t), C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p,
                                    C.c_void_p, C.c_size_t, C.POINTER(cuth_import_report_t), C.c_void_p]
    rc = L.cuth_import_csr_n(grid.ref(), _ptr(rowptr), _ptr(col), _ptr(val),
                             C.c_int64(val.numel() if nnz is None else int(nnz)),
                             None if rs is None else rs.ctypes.data_as(C.c_void_p), _ptr(dia),
                             dia.numel() * dia.element_size(), C.byref(rep), stream or _stream())
    if not check:
        return rc, rep
    _check(rc, "cuth_import_csr")
    return rep


def cuth_import_coo(grid: Grid, row, col, val, dia, rowsum_layer=None, stream=None, check=True):
    """row, col int32 / val float64 CUDA tensors of equal length (any order).  As cuth_import_csr."""
    import torch
    assert row.dtype == torch.int32 and col.dtype == torch.int32 and val.dtype == torch.float64
    assert row.numel() == col.numel() == val.numel()
    rep = cuth_import_report_t()
    rs = None if rowsum_layer is None else np.ascontiguousarray(rowsum_layer, dtype=np.float64)
    rc = load_library().cuth_import_coo(grid.ref(), _ptr(row), _ptr(col), _ptr(val), C.c_int64(val.numel()),
                                        None if rs is None else rs.ctypes.data_as(C.c_void_p), _ptr(dia),
                                        dia.numel() * dia.element_size(), C.byref(rep), stream or _stream())
    if not check:
        return rc, rep
    _check(rc, "cuth_import_coo")
    return rep


def cuth_dia_view(dia, grid: Grid):
    """Returns (vals_ptr, vals32_ptr, inv_diag_ptr, ptr[5], off[4]); pointers are device addresses."""
    v, v32, dinv = C.c_void_p(), C.c_void_p(), C.c_void_p()
    ptr = (C.c_int64 * 5)()
    off = (C.c_int64 * 4)()
    _check(load_library().cuth_dia_view(_ptr(dia), grid.ref(), C.byref(v), C.byref(v32), C.byref(dinv), ptr, off),
           "cuth_dia_view")
    return v.value, v32.value, dinv.value, list(ptr), list(off)


def cuth_spmv(dia, grid: Grid, precision, x, y, stream=None):
    _check(load_library().cuth_spmv(_ptr(dia), grid.ref(), int(precision), _ptr(x), _ptr(y), stream or _stream()),
           "cuth_spmv")


def cuth_spmv_tuned(dia, grid: Grid, precision, tuning, x, y, stream=None):
    t = tuning if tuning is not None else Tuning()
    _check(load_library().cuth_spmv_tuned(_ptr(dia), grid.ref(), int(precision), C.byref(t), _ptr(x), _ptr(y),
                                          stream or _stream()), "cuth_spmv_tuned")


def cuth_pcg_solve(dia, grid: Grid, opts, b, x, work, result, stream=None):
    _check(load_library().cuth_pcg_solve(_ptr(dia), grid.ref(), C.byref(opts), _ptr(b), _ptr(x), _ptr(work),
                                         work.numel() * work.element_size(), _ptr(result), stream or _stream()),
           "cuth_pcg_solve")


def cuth_batch_workspace_bytes(grid: Grid, nrhs: int) -> int:
    return int(load_library().cuth_batch_workspace_bytes(grid.ref(), int(nrhs)))


def cuth_pcg_solve_batch(dia, grid: Grid, opts, nrhs, b, x, work, result, stream=None):
    """b, x: [nrhs, N] float64 CUDA tensors (contiguous); result: device buffer of nrhs cuth_result_t records."""
    _check(load_library().cuth_pcg_solve_batch(_ptr(dia), grid.ref(), C.byref(opts), int(nrhs), _ptr(b), _ptr(x),
                                               _ptr(work), work.numel() * work.element_size(), _ptr(result),
                                               stream or _stream()), "cuth_pcg_solve_batch")


def cuth_transient_step(dia, grid: Grid, opts, power, T, work, result, stream=None):
    _check(load_library().cuth_transient_step(_ptr(dia), grid.ref(), C.byref(opts), _ptr(power), _ptr(T), _ptr(work),
                                              work.numel() * work.element_size(), _ptr(result),
                                              stream or _stream()), "cuth_transient_step")


def cuth_release_workspace(work):
    load_library().cuth_release_workspace(_ptr(work))


def cuth_profile_kernel(work, grid: Grid, opts, kernel_id: int, stream=None):
    _check(load_library().cuth_profile_kernel(_ptr(work), grid.ref(), C.byref(opts), int(kernel_id),
                                              stream or _stream()), "cuth_profile_kernel")


def cuth_lanczos_bounds(dia, grid: Grid, v0, steps, work, stream=None, tuning=None):
    """Returns (ritz_min, ritz_max, gershgorin_max, lmin, lmax); synchronises the stream."""
    out = (C.c_double * 5)()
    t = tuning if tuning is not None else Tuning()
    _check(load_library().cuth_lanczos_bounds_tuned(_ptr(dia), grid.ref(), C.byref(t), _ptr(v0), int(steps),
                                                    _ptr(work), work.numel() * work.element_size(), out,
                                                    stream or _stream()), "cuth_lanczos_bounds")
    return tuple(out)


def cuth_policy_probe(rr, tt, dd, tt_prev, rr_prev, bb, rtol, soft_drift=0.0, late=False, conv_rec=False,
                      capped=False):
    """The device-side decision after one evaluation of r_true (include/cuth.h cuth_policy_probe) on SQUARED norms;
    returns dict(go, stage, switch_reason, switch_mask, restart, status, promotions).  Synchronises."""
    import torch
    vals = (C.c_double * 8)(float(rr), float(tt), float(dd), float(tt_prev), float(rr_prev), float(bb), float(rtol),
                            float(soft_drift))
    out = torch.zeros(8, dtype=torch.int32, device="cuda")
    flags = (1 if late else 0) | (2 if conv_rec else 0) | (4 if capped else 0)
    _check(load_library().cuth_policy_probe(vals, flags, _ptr(out), _stream()), "cuth_policy_probe")
    o = out.cpu().tolist()
    return dict(go=o[0], stage=o[1], switch_reason=o[2], switch_mask=o[3], restart=o[4], status=o[5], promotions=o[6])


def cuth_cheb_apply(dia, grid: Grid, opts, r, z, work, stream=None):
    _check(load_library().cuth_cheb_apply(_ptr(dia), grid.ref(), C.byref(opts), _ptr(r), _ptr(z), _ptr(work),
                                          work.numel() * work.element_size(), stream or _stream()), "cuth_cheb_apply")


def cuth_tridiag_extremes(alpha, beta):
    a = np.ascontiguousarray(alpha, dtype=np.float64)
    b = np.ascontiguousarray(beta, dtype=np.float64)
    out = (C.c_double * 2)()
    L = load_library()
    L.cuth_tridiag_extremes.restype = C.c_int
    _check(L.cuth_tridiag_extremes(a.ctypes.data_as(C.c_void_p), b.ctypes.data_as(C.c_void_p), C.c_int(a.size), out),
           "cuth_tridiag_extremes")
    return out[0], out[1]


def cuth_cheb_launches(grid: Grid, opts):
    """(launches, pairs) of one Chebyshev apply for this grid and these options (include/cuth.h); pure host."""
    L = load_library()
    L.cuth_cheb_launches.restype = C.c_int
    pairs = C.c_int(0)
    rc = L.cuth_cheb_launches(grid.ref(), C.byref(opts), C.byref(pairs))
    if rc < 0:
        _check(rc, "cuth_cheb_launches")
    return int(rc), int(pairs.value)


def cuth_version() -> int:
    return int(load_library().cuth_version())


def cuth_noalloc_max_rows() -> int:
    L = load_library()
    L.cuth_noalloc_max_rows.restype = C.c_int64
    return int(L.cuth_noalloc_max_rows())


def cuth_residual_noalloc(dia, grid: Grid, b, x, out, t=None, stream=None, check=True):
    """t = b - A1 x, out[0..3] = ||t||^2, ||b||^2, ||t|| / ||b||, 0 -- without any workspace (include/cuth.h).  `out`: CUDA
    float64 tensor of >= 4 elements.  Raises CuthError (with the library's message) unless check=False (returns rc)."""
    L = load_library()
    L.cuth_residual_noalloc.restype = C.c_int
    L.cuth_residual_noalloc.argtypes = [C.c_void_p, C.POINTER(cuth_grid_t), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p]
    L.cuth_noalloc_last_error.restype = C.c_char_p
    rc = L.cuth_residual_noalloc(_ptr(dia), grid.ref(), _ptr(b), _ptr(x), _ptr(t), _ptr(out), stream or _stream())
    if not check:
        return rc
    if rc != 0:
        e = CuthError(rc, "cuth_residual_noalloc")
        e.args = (e.args[0] + ": " + L.cuth_noalloc_last_error().decode(),)
        raise e
    return rc


def cuth_loop_home(grid: Grid, opts) -> int:
    """1 graph, 2 persistent kernel, 3 cluster-resident kernel, 4 fixed-FP32 kernel (include/cuth.h); pure host."""
    L = load_library()
    L.cuth_loop_home.restype = C.c_int
    L.cuth_loop_home.argtypes = [C.POINTER(cuth_grid_t), C.POINTER(cuth_opts_t)]
    rc = int(L.cuth_loop_home(grid.ref(), C.byref(opts)))
    if rc < 0:
        _check(rc, "cuth_loop_home")
    return rc


def cuth_traversal(grid: Grid, opts) -> int:
    """1 flat, 2 z-marching (include/cuth.h); pure host."""
    L = load_library()
    L.cuth_traversal.restype = C.c_int
    L.cuth_traversal.argtypes = [C.POINTER(cuth_grid_t), C.POINTER(cuth_opts_t)]
    rc = int(L.cuth_traversal(grid.ref(), C.byref(opts)))
    if rc < 0:
        _check(rc, "cuth_traversal")
    return rc


def cuth_launches_per_iteration(grid: Grid, opts) -> int:
    return int(load_library().cuth_launches_per_iteration(grid.ref(), C.byref(opts)))


# ------------------------------------------------------------------ convenience holders (allocation only)
class DiaMatrix:
    """Allocates the matrix buffer with torch and calls cuth_build_dia (or, with csr=(rowptr, col, val) CUDA
    tensors, cuth_import_csr)."""

    def __init__(self, grid: Grid, csr=None, rowsum_layer=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("cuth needs a CUDA device (no CPU fallback)")
        self.grid = grid
        nbytes = cuth_dia_bytes(grid)
        if nbytes == 0:
            raise CuthError(-2, "cuth_dia_bytes")
        self.buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.import_report = None
        if csr is None:
            cuth_build_dia(grid, self.buf)
        else:
            self.import_report = cuth_import_csr(grid, csr[0], csr[1], csr[2], self.buf, rowsum_layer)

    def view(self):
        """(vals fp64 [E], vals32 fp32 [E], inv_diag fp64 [N], ptr, off) as torch views of the buffer."""
        import torch
        v, v32, dinv, ptr, off = cuth_dia_view(self.buf, self.grid)
        base = self.buf.data_ptr()
        e = ptr[4]
        vals = self.buf[v - base: v - base + 8 * e].view(torch.float64)
        vals32 = self.buf[v32 - base: v32 - base + 4 * e].view(torch.float32)
        inv = self.buf[dinv - base: dinv - base + 8 * self.grid.n].view(torch.float64)
        return vals, vals32, inv, ptr, off

    def spmv(self, x, precision=FP64, out=None):
        import torch
        y = torch.empty_like(x) if out is None else out
        cuth_spmv_tuned(self.buf, self.grid, precision, None, x, y)
        return y


class BatchSolver:
    """Workspace + result records for cuth_pcg_solve_batch (allocation only)."""

    def __init__(self, A: "DiaMatrix", nrhs: int, opts=None):
        import torch
        self.A, self.nrhs = A, int(nrhs)
        self.opts = opts or Opts()
        nbytes = cuth_batch_workspace_bytes(A.grid, self.nrhs)
        if nbytes == 0:
            raise CuthError(-3, "cuth_batch_workspace_bytes")
        self.work = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.result_dev = torch.zeros(self.nrhs * C.sizeof(cuth_result_t), dtype=torch.uint8, device="cuda")

    def solve(self, b, x):
        assert b.is_contiguous() and x.is_contiguous() and b.shape == x.shape == (self.nrhs, self.A.grid.n)
        cuth_pcg_solve_batch(self.A.buf, self.A.grid, self.opts, self.nrhs, b, x, self.work, self.result_dev)

    def results(self):
        """Synchronising read-back of the nrhs device result records."""
        raw = self.result_dev.cpu().numpy().tobytes()
        sz = C.sizeof(cuth_result_t)
        out = []
        for s in range(self.nrhs):
            r = cuth_result_t.from_buffer_copy(raw[s * sz:(s + 1) * sz])
            out.append(Result(r.status, r.iterations, r.promotions, r.true_resid_evals, r.rel_resid_true,
                              r.rel_resid_rec, r.switch_reason, r.switch_iteration, r.switch_mask, r.hard_restarts,
                              r.soft_restarts))
        return out


class Solver:
    """Allocates workspace + result record once; solve()/step() enqueue without synchronising."""

    def __init__(self, A: DiaMatrix, opts=None):
        import torch
        self.A = A
        self.opts = opts or Opts()
        self.work = torch.empty(cuth_workspace_bytes(A.grid, self.opts), dtype=torch.uint8, device="cuda")
        self.result_dev = torch.zeros(C.sizeof(cuth_result_t), dtype=torch.uint8, device="cuda")

    def setup_chebyshev(self, v0, lanczos_steps=40, degree=30, lmin=None, lmax=None, storage=CHEB_DEFAULT):
        """Spectral range by Lanczos (cuth_lanczos_bounds) and switch this solver to the Chebyshev
        preconditioner; only copies the interval the library returns into the options struct."""
        import torch
        lo, hi, gersh, rec_lo, rec_hi = cuth_lanczos_bounds(self.A.buf, self.A.grid, v0, lanczos_steps, self.work,
                                                            tuning=self.opts.tuning)
        o = self.opts
        self.opts = Opts(o.precision, o.rtol, o.max_iters, o.true_resid_period, PRECOND_CHEBYSHEV, degree,
                         rec_lo if lmin is None else lmin, rec_hi if lmax is None else lmax, storage, o.tuning)
        need = cuth_workspace_bytes(self.A.grid, self.opts)
        if need > self.work.numel():
            cuth_release_workspace(self.work)
            self.work = torch.empty(need, dtype=torch.uint8, device="cuda")
        return lo, hi, gersh

    def cheb_apply(self, r, z):
        cuth_cheb_apply(self.A.buf, self.A.grid, self.opts, r, z, self.work)

    def solve(self, b, x):
        cuth_pcg_solve(self.A.buf, self.A.grid, self.opts, b, x, self.work, self.result_dev)

    def step(self, power, T):
        cuth_transient_step(self.A.buf, self.A.grid, self.opts, power, T, self.work, self.result_dev)

    def result(self) -> Result:
        """Synchronising read-back of the device result record."""
        raw = self.result_dev.cpu().numpy().tobytes()
        r = cuth_result_t.from_buffer_copy(raw)
        return Result(r.status, r.iterations, r.promotions, r.true_resid_evals, r.rel_resid_true,
                      r.rel_resid_rec, r.switch_reason, r.switch_iteration, r.switch_mask, r.hard_restarts,
                      r.soft_restarts)

    def close(self):
        cuth_release_workspace(self.work)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
