"""Pins of the oracle's 7-point structure checker (oracle.stencil7_report; SURVEY.md §8(f) importer) against
matrices whose defects are planted by hand, so the expected counts are known without running it, and against
scipy's own symmetry / bandwidth facts."""
import numpy as np
import scipy.sparse as sp

import workloads as W
from oracle import oracle as O
from import_faults import faults

EXPECTED = {   # name: (off_stencil, asymmetric_rows, bad_diagonal, duplicates)
    "off_stencil_pair": (2, 0, 0, 0),
    "wrap_x": (2, 0, 0, 0),
    "wrap_y": (2, 0, 0, 0),
    "asymmetric": (0, 1, 0, 0),
    "negative_diagonal": (0, 0, 1, 0),
    "duplicate": (0, 0, 0, 1),
    "explicit_zero_off_stencil": (0, 0, 0, 0),
    "column_out_of_range": (1, 0, 0, 0),
}


def test_assembled_matrices_pass_and_row_sums_are_the_physical_ones():
    for kw in (dict(cfg=1, nx=4, ny=3, nz=2, n_hot=1), dict(cfg=3, nx=9, ny=7, nz=5, n_hot=2),
               dict(cfg=5, nx=8, ny=6, nz=4, n_hot=2), dict(cfg=6, nx=7, ny=5, nz=10, n_hot=2)):
        w = W.make_workload(**kw)
        A = O.assemble_workload(w)
        rep = O.stencil7_report(A, w.nx, w.ny, w.nz)
        assert (rep["off_stencil"], rep["asymmetric_rows"], rep["bad_diagonal"], rep["duplicates"],
                rep["positive_offdiag"]) == (0, 0, 0, 0, 0)
        assert rep["mixed_ok"] == 1
        # eq. (4)/(5): conductances cancel in a row sum; what is left is the Robin term on
        # the top layer and C V / dt everywhere
        s = np.zeros(w.nz)
        s[-1] += w.h_top * w.dx * w.dy
        if w.cvol is not None and w.dt > 0:
            s += np.asarray(w.cvol) * w.dx * w.dy * np.asarray(w.dz) / w.dt
        dmin = A.to_scipy().diagonal().min()
        assert np.abs(rep["s_layer"] - s).max() <= 1e-12 * dmin
        # independent facts from scipy: symmetric, and every non-zero on one of the seven offsets
        M = A.to_scipy()
        assert (M - M.T).nnz == 0
        coo = M.tocoo()
        assert set(np.unique(coo.col - coo.row)) <= {0, 1, -1, w.nx, -w.nx, w.nx * w.ny, -w.nx * w.ny}


def test_planted_defects_are_counted():
    w = W.make_workload(cfg=3, nx=12, ny=9, nz=5, n_hot=2)
    A = O.assemble_workload(w)
    fs = faults(A, w.nx, w.ny, w.nz)
    assert set(fs) == set(EXPECTED)
    for name, Af in fs.items():
        rep = O.stencil7_report(Af, w.nx, w.ny, w.nz)
        got = (rep["off_stencil"], rep["asymmetric_rows"], rep["bad_diagonal"], rep["duplicates"])
        assert got == EXPECTED[name], name


def test_wrap_entries_are_what_a_plain_band_check_misses():
    """The planted x-wrap entry sits ON offset +1, so a bandwidth check passes it; only the cell geometry rejects it."""
    w = W.make_workload(cfg=1, nx=5, ny=4, nz=3, n_hot=1)
    A = O.assemble_workload(w)
    Af = faults(A, w.nx, w.ny, w.nz)["wrap_x"]
    coo = sp.csr_matrix((Af.val, Af.col, Af.rowptr), shape=(Af.n, Af.n)).tocoo()
    assert set(np.unique(coo.col - coo.row)) <= {0, 1, -1, w.nx, -w.nx, w.nx * w.ny, -w.nx * w.ny}
    assert O.stencil7_report(Af, w.nx, w.ny, w.nz)["off_stencil"] == 2


def test_non_layered_diagonal_shift_is_flagged():
    w = W.make_workload(cfg=3, nx=9, ny=7, nz=5, n_hot=2)
    A = O.assemble_workload(w)
    rows = np.repeat(np.arange(A.n), np.diff(A.rowptr))
    v = A.val.copy()
    dq = np.flatnonzero(A.col == rows)
    shift = 0.05 * W.uniform01(w.seed, 77, np.arange(A.n))
    v[dq] *= 1.0 + shift
    rep = O.stencil7_report(O.CSR(A.n, A.rowptr, A.col, v), w.nx, w.ny, w.nz)
    assert rep["mixed_ok"] == 0 and rep["off_stencil"] == rep["asymmetric_rows"] == rep["bad_diagonal"] == 0
    # the row sums are now shift_i * D0_i (+ s): the deviation is at least half their spread over the smallest diagonal
    d = A.val[dq]
    spread = (shift * d).reshape(w.nz, -1)
    lower = max((r.max() - r.min()) / 2 / (dd.min() * 1.05) for r, dd in zip(spread, d.reshape(w.nz, -1)))
    assert rep["max_rowsum_dev"] >= 0.9 * lower
