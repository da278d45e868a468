"""CSR matrices with one planted defect each, for the importer tests (CPU pin of the oracle's checker and the GPU
comparison).  Inputs only: no arithmetic of the method lives here."""
import numpy as np

from oracle import oracle as O


def with_entries(A, extra_rows, extra_cols, extra_vals):
    """A plus extra entries appended to their rows (CSR rebuilt by hand; nothing is summed)."""
    rows = np.repeat(np.arange(A.n), np.diff(A.rowptr))
    rows = np.concatenate([rows, np.asarray(extra_rows, dtype=np.int64)])
    cols = np.concatenate([A.col, np.asarray(extra_cols, dtype=np.int32)])
    vals = np.concatenate([A.val, np.asarray(extra_vals, dtype=np.float64)])
    order = np.argsort(rows, kind="stable")
    rowptr = np.zeros(A.n + 1, dtype=np.int64)
    np.add.at(rowptr, rows + 1, 1)
    return O.CSR(A.n, np.cumsum(rowptr), cols[order].astype(np.int32), vals[order])


def faults(A, nx, ny, nz):
    n, nxny = A.n, nx * ny
    rows = np.repeat(np.arange(n), np.diff(A.rowptr))
    out = {}
    out["off_stencil_pair"] = with_entries(A, [0, 2 + nx], [2 + nx, 0], [-1e-7, -1e-7])      # offset nx + 2: not a diagonal
    i = nx - 1                                                                        # x = nx-1 -> x = 0 of the next line
    out["wrap_x"] = with_entries(A, [i, i + 1], [i + 1, i], [-1e-7, -1e-7])
    i = nx * (ny - 1) + 1                                                             # y = ny-1 -> y = 0 of the next plane
    out["wrap_y"] = with_entries(A, [i, i + nx], [i + nx, i], [-1e-7, -1e-7])
    v = A.val.copy()
    q = np.flatnonzero((A.col - rows) == -nx)[3]
    v[q] *= 1.0 + 1e-12
    out["asymmetric"] = O.CSR(n, A.rowptr, A.col, v)
    v = A.val.copy()
    q = np.flatnonzero((A.col - rows) == 0)[5]
    v[q] = -v[q]
    out["negative_diagonal"] = O.CSR(n, A.rowptr, A.col, v)
    out["duplicate"] = with_entries(A, [3], [3 + nxny], [-1e-7])
    out["explicit_zero_off_stencil"] = with_entries(A, [0], [n - 1], [0.0])                  # harmless
    out["column_out_of_range"] = with_entries(A, [n - 1], [n], [-1e-7])
    return out
