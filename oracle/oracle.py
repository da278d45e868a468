"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_2606_17850_b200.
Each function is a thin call into oracle/cuth_oracle.cpp, whose header cites the
passages of the paper it follows.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_csr_nnz.restype = C.c_int64
        _lib.oracle_csr_nnz.argtypes = [C.c_int64] * 3
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def num_threads() -> int:
    return int(lib().oracle_num_threads())


@dataclass
class CSR:
    n: int
    rowptr: np.ndarray   # int64 [n+1]
    col: np.ndarray      # int32 [nnz]
    val: np.ndarray      # float64 [nnz]

    def to_scipy(self):
        import scipy.sparse as sp
        return sp.csr_matrix((self.val, self.col, self.rowptr), shape=(self.n, self.n))


def assemble_csr(nx, ny, nz, dx, dy, dz, kappa, h_top, cvol=None, dt=0.0) -> CSR:
    """eq. (4)/(5) -> CSR.  kappa: nz values (layered) or nx*ny*nz values (per cell)."""
    L = lib()
    n = nx * ny * nz
    dz = np.ascontiguousarray(dz, dtype=np.float64)
    kappa = np.ascontiguousarray(kappa, dtype=np.float64)
    assert dz.size == nz and kappa.size in (nz, n)
    per_layer = 1 if kappa.size == nz and nz != n else 0
    if kappa.size == nz and nz == n:
        per_layer = 1
    cv = None if cvol is None else np.ascontiguousarray(cvol, dtype=np.float64)
    nnz = int(L.oracle_csr_nnz(nx, ny, nz))
    rowptr = np.empty(n + 1, dtype=np.int64)
    col = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float64)
    rc = L.oracle_assemble_csr(C.c_int64(nx), C.c_int64(ny), C.c_int64(nz), C.c_double(dx), C.c_double(dy),
                               _p(dz), _p(kappa), C.c_int(per_layer), C.c_double(h_top), _p(cv),
                               C.c_double(dt), _p(rowptr), _p(col), _p(val))
    assert rc == 0 and rowptr[-1] == nnz
    return CSR(n, rowptr, col, val)


def assemble_workload(w) -> CSR:
    kappa = w.kappa_cell if w.kappa_cell is not None else w.kappa_layer
    return assemble_csr(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, kappa, w.h_top, w.cvol, w.dt)


def spmv(A: CSR, x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty(A.n, dtype=np.float64)
    lib().oracle_csr_spmv(C.c_int64(A.n), _p(A.rowptr), _p(A.col), _p(A.val), _p(x), _p(y))
    return y


def csr_to_dia(A: CSR, nx, ny, nz):
    """Condensed DIA: returns vals[E], ptr[5], off[4]."""
    n = nx * ny * nz
    e = 4 * n - 1 - nx - nx * ny
    vals = np.empty(e, dtype=np.float64)
    ptr = np.empty(5, dtype=np.int64)
    off = np.empty(4, dtype=np.int64)
    lib().oracle_csr_to_dia(C.c_int64(nx), C.c_int64(ny), C.c_int64(nz), _p(A.rowptr), _p(A.col), _p(A.val),
                            _p(vals), _p(ptr), _p(off))
    assert ptr[4] == e
    return vals, ptr, off


def stencil7_report(A: CSR, nx, ny, nz) -> dict:
    """Is this CSR matrix a symmetric 7-point matrix of the nx x ny x nz box?  The definition written out entry by
    entry (SURVEY.md §8(f) importer; the diagonals are those of PAPER.md:219 / Alg. 2):
    an entry (i, j) is ON the stencil when j - i is one of {0, +-1, +-nx, +-nx*ny}, 0 <= j < n, and a +-1 / +-nx
    step stays inside the line / plane of cell i.  Counts: non-zero entries off the stencil; repeats of an on-stencil
    (i, j); rows whose first diagonal entry is missing, <= 0 or not finite; rows where a lower on-stencil entry
    differs from its mirror (absent == 0); on-stencil off-diagonal entries > 0; and the largest deviation of a row
    sum from the midrange row sum of its layer, relative to the layer's smallest diagonal entry."""
    n = nx * ny * nz
    nxny = nx * ny
    first = {}
    off_stencil = duplicates = positive = 0
    for i in range(n):
        x, y = i % nx, (i % nxny) // nx
        for q in range(int(A.rowptr[i]), int(A.rowptr[i + 1])):
            j, v = int(A.col[q]), float(A.val[q])
            c = j - i
            on = 0 <= j < n and c in (0, 1, -1, nx, -nx, nxny, -nxny)
            if on and c == 1:
                on = x + 1 < nx
            if on and c == -1:
                on = x > 0
            if on and c == nx:
                on = y + 1 < ny
            if on and c == -nx:
                on = y > 0
            if not on:
                off_stencil += 1 if v != 0.0 else 0
                continue
            if (i, j) in first:
                duplicates += 1
                continue
            first[(i, j)] = v
            if c != 0 and v > 0.0:
                positive += 1
    bad_diagonal = sum(1 for i in range(n) if not (first.get((i, i), 0.0) > 0.0 and np.isfinite(first[(i, i)])))
    asymmetric_rows = 0
    rowsum = np.zeros(n)
    for i in range(n):
        bad = False
        rs = first.get((i, i), 0.0)
        for o in (nxny, nx, 1):
            if i - o >= 0:
                bad = bad or first.get((i, i - o), 0.0) != first.get((i - o, i), 0.0)
                rs += first.get((i - o, i), 0.0)
        for o in (1, nx, nxny):
            if i + o < n:
                rs += first.get((i, i + o), 0.0)
        asymmetric_rows += 1 if bad else 0
        rowsum[i] = rs
    dev = 0.0
    s_layer = np.zeros(nz)
    for z in range(nz):
        rs = rowsum[z * nxny:(z + 1) * nxny]
        d = np.array([first.get((i, i), 0.0) for i in range(z * nxny, (z + 1) * nxny)])
        s = max(0.0, 0.5 * (rs.min() + rs.max()))
        s_layer[z] = s
        dmin = d.min() if d.min() > 0 else 1.0
        dev = max(dev, max(abs(rs.max() - s), abs(rs.min() - s)) / dmin)
    ok = off_stencil == 0 and duplicates == 0 and bad_diagonal == 0 and asymmetric_rows == 0
    return dict(off_stencil=off_stencil, asymmetric_rows=asymmetric_rows, bad_diagonal=bad_diagonal,
                duplicates=duplicates, positive_offdiag=positive, max_rowsum_dev=dev,
                mixed_ok=int(ok and dev <= 1e-9), s_layer=s_layer)


def transient_rhs(w, power: np.ndarray, t_n: np.ndarray) -> np.ndarray:
    b = np.empty(w.n, dtype=np.float64)
    power = np.ascontiguousarray(power, dtype=np.float64)
    t_n = np.ascontiguousarray(t_n, dtype=np.float64)
    lib().oracle_transient_rhs(C.c_int64(w.nx), C.c_int64(w.ny), C.c_int64(w.nz), C.c_double(w.dx),
                               C.c_double(w.dy), _p(np.ascontiguousarray(w.dz)), _p(np.ascontiguousarray(w.cvol)),
                               C.c_double(w.dt), _p(power), _p(t_n), _p(b))
    return b


@dataclass
class PCGResult:
    x: np.ndarray
    status: int          # 0 converged, 1 max_iters, 2 breakdown
    iterations: int
    rel_resid_true: float
    hist: np.ndarray | None = None


def pcg(A: CSR, b, x0=None, rtol=1e-8, max_iters=200000, precond=1, hist_len=0) -> PCGResult:
    """Alg. 1 with M = diag(A) (precond=1) or I (precond=0)."""
    b = np.ascontiguousarray(b, dtype=np.float64)
    x = np.zeros(A.n, dtype=np.float64) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    it = C.c_int64(0)
    rel = C.c_double(0.0)
    hist = np.full(hist_len, np.nan) if hist_len > 0 else None
    st = lib().oracle_pcg(C.c_int64(A.n), _p(A.rowptr), _p(A.col), _p(A.val), _p(b), _p(x), C.c_double(rtol),
                          C.c_int64(max_iters), C.c_int(precond), C.byref(it), C.byref(rel), _p(hist),
                          C.c_int64(hist_len))
    return PCGResult(x, int(st), int(it.value), float(rel.value), hist)


def pcg_window(A: CSR, b, x0, iters: int, precond=1) -> np.ndarray:
    """Exactly `iters` iterations of Alg. 1 (timing windows on grids too big for a full CPU solve)."""
    b = np.ascontiguousarray(b, dtype=np.float64)
    x = np.array(x0, dtype=np.float64, copy=True)
    lib().oracle_pcg_window(C.c_int64(A.n), _p(A.rowptr), _p(A.col), _p(A.val), _p(b), _p(x),
                            C.c_int64(iters), C.c_int(precond))
    return x


# ------------------------------------------------------------------ NEXT-1: Chebyshev + Lanczos
def cheb_apply(A: CSR, r, lmin, lmax, k) -> np.ndarray:
    """Alg. 3: z = q(A) r, degree-k Chebyshev preconditioner on [lmin, lmax]."""
    r = np.ascontiguousarray(r, dtype=np.float64)
    z = np.empty(A.n, dtype=np.float64)
    lib().oracle_cheb_apply(C.c_int64(A.n), _p(A.rowptr), _p(A.col), _p(A.val), _p(r), C.c_double(lmin),
                            C.c_double(lmax), C.c_int(k), _p(z))
    return z


def lanczos(A: CSR, v0, m):
    """m Lanczos steps: returns alpha[m'], beta[m'] of the tridiagonal T (m' <= m)."""
    v0 = np.ascontiguousarray(v0, dtype=np.float64)
    alpha = np.zeros(m)
    beta = np.zeros(m)
    done = lib().oracle_lanczos(C.c_int64(A.n), _p(A.rowptr), _p(A.col), _p(A.val), _p(v0), C.c_int(m),
                                _p(alpha), _p(beta))
    return alpha[:done], beta[:done]


def ritz_extremes(alpha, beta):
    """Extreme eigenvalues of T = tridiag(beta[:-1], alpha, beta[:-1]) (host, fp64, LAPACK)."""
    import scipy.linalg as sla
    w = sla.eigvalsh_tridiagonal(np.asarray(alpha), np.asarray(beta[:len(alpha) - 1]))
    return float(w[0]), float(w[-1])


def pcg_cheb(A: CSR, b, lmin, lmax, k, x0=None, rtol=1e-8, max_iters=200000) -> PCGResult:
    """Alg. 1 with M^-1 = Alg. 3."""
    b = np.ascontiguousarray(b, dtype=np.float64)
    x = np.zeros(A.n, dtype=np.float64) if x0 is None else np.array(x0, dtype=np.float64, copy=True)
    it = C.c_int64(0)
    rel = C.c_double(0.0)
    st = lib().oracle_pcg_cheb(C.c_int64(A.n), _p(A.rowptr), _p(A.col), _p(A.val), _p(b), _p(x), C.c_double(rtol),
                               C.c_int64(max_iters), C.c_double(lmin), C.c_double(lmax), C.c_int(k),
                               C.byref(it), C.byref(rel))
    return PCGResult(x, int(st), int(it.value), float(rel.value))
