"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

A plausible mistake anywhere in oracle/cuth_oracle.cpp (dropped term, wrong sign or index,
transposed operand, wrong diagonal offset) must fail at least one of these.
Citations: eq. (4), 130-133 eq. (5), 137 (SPD, seven diagonals), 145-168 Alg. 1,
192-215 Alg. 2, 219 (Quad-Diag), Table I 420-428 (NNZ/N).
"""
import os

import numpy as np
import pytest
import scipy.linalg as sla

import workloads as W
from oracle import oracle as O
from direct_solve import solve_layered

HERE = os.path.dirname(os.path.abspath(__file__))
TINY = [(4, 3, 2), (5, 4, 3), (7, 2, 5), (2, 2, 2)]


def _rand_problem(nx, ny, nz, seed, per_cell=True, transient=False):
    n = nx * ny * nz
    idx = np.arange(n)
    dz = 1e-6 * (0.5 + W.uniform01(seed, 11, np.arange(nz)))
    if per_cell:
        kappa = 1.0 + 300.0 * W.uniform01(seed, 12, idx)
    else:
        kappa = 1.0 + 300.0 * W.uniform01(seed, 12, np.arange(nz))
    cvol = (1e6 * (1.0 + W.uniform01(seed, 13, np.arange(nz)))) if transient else None
    dt = 1e-5 if transient else 0.0
    dx, dy, h = 1.3e-6, 0.7e-6, 1.0e4
    A = O.assemble_csr(nx, ny, nz, dx, dy, dz, kappa, h, cvol, dt)
    b = 1e-6 * W.uniform01(seed, 14, idx)
    return A, b, dict(dx=dx, dy=dy, dz=dz, kappa=kappa, h=h, cvol=cvol, dt=dt)


# ---------------------------------------------------------------- structure and invariants
@pytest.mark.parametrize("dims", TINY + [(32, 32, 8)])
def test_nnz_closed_form_and_table1_ratio(dims):
    nx, ny, nz = dims
    A, _, _ = _rand_problem(nx, ny, nz, 1, per_cell=False)
    n = nx * ny * nz
    assert A.val.size == 7 * n - 2 * (nx * ny + nx * nz + ny * nz)
    if dims == (32, 32, 8):
        assert A.val.size == 54272          # SURVEY.md §4 probe value


def test_table1_nnz_over_n():
    # Table I: NNZ/N = 3.4e7/5.1e6 ... 2.3e8/3.5e7 = 6.57..6.79 at nz = 10
    nx = ny = 714   # 714^2 * 10 = 5.1e6 (CUTh1)
    ratio = (7 * nx * ny * 10 - 2 * (nx * ny + 2 * nx * 10)) / (nx * ny * 10)
    assert 6.5 < ratio < 6.85


@pytest.mark.parametrize("dims", TINY)
@pytest.mark.parametrize("transient", [False, True])
def test_invariants_symmetry_signs_rowsums(dims, transient):
    nx, ny, nz = dims
    A, _, p = _rand_problem(nx, ny, nz, 2, per_cell=True, transient=transient)
    M = A.to_scipy().toarray()
    n = nx * ny * nz
    assert np.array_equal(M, M.T)                      # bitwise symmetric (same g both sides)
    assert np.all(np.diag(M) > 0)
    off = M - np.diag(np.diag(M))
    assert np.all(off <= 0)
    # only offsets 0, +-1, +-nx, +-nx*ny carry entries
    ii, jj = np.nonzero(M)
    assert set(np.abs(ii - jj).tolist()) <= {0, 1, nx, nx * ny}
    # row sums: A 1 = s, s = h dx dy on the top layer (+ C V / dt)   (eq. (4)/(5))
    s = np.zeros((nz, ny, nx))
    s[nz - 1] += p["h"] * p["dx"] * p["dy"]
    if transient:
        s += (p["cvol"] * p["dx"] * p["dy"] * p["dz"] / p["dt"])[:, None, None]
    rs = O.spmv(A, np.ones(n))
    assert np.allclose(rs, s.reshape(-1), rtol=0, atol=1e-12 * np.abs(np.diag(M)).max())
    # SPD
    w = np.linalg.eigvalsh(M)
    assert w.min() > 0


def test_no_wraparound_coupling():
    # cell x = nx-1 must not couple to x = 0 of the next row (offset +1 across a row end)
    nx, ny, nz = 5, 4, 3
    A, _, _ = _rand_problem(nx, ny, nz, 3)
    M = A.to_scipy().toarray()
    for z in range(nz):
        for y in range(ny):
            i = (nx - 1) + nx * (y + ny * z)
            if i + 1 < nx * ny * nz:
                assert M[i, i + 1] == 0.0
        i = nx * (ny - 1) + nx * ny * z      # y = ny-1 must not couple to y = 0 of next plane
        if i + nx < nx * ny * nz:
            assert M[i, i + nx] == 0.0


def test_conductance_values_against_hand_formula():
    # 2x2x2, distinct kappas: check three entries against eq. (4) conductances typed by hand
    k = np.array([10., 20., 30., 40., 50., 60., 70., 80.])
    dx, dy, dz = 2e-6, 3e-6, np.array([1e-6, 4e-6])
    A = O.assemble_csr(2, 2, 2, dx, dy, dz, k, 1e4)
    M = A.to_scipy().toarray()
    g01 = dy * dz[0] / (dx / 20. + dx / 40.)               # cells 0,1 (x neighbours, z=0)
    g02 = dx * dz[0] / (dy / 20. + dy / 60.)               # cells 0,2 (y neighbours)
    g04 = dx * dy / (dz[0] / 20. + dz[1] / 100.)           # cells 0,4 (z neighbours)
    assert M[0, 1] == pytest.approx(-g01, rel=1e-15)
    assert M[0, 2] == pytest.approx(-g02, rel=1e-15)
    assert M[0, 4] == pytest.approx(-g04, rel=1e-15)
    assert M[0, 0] == pytest.approx(g01 + g02 + g04, rel=1e-15)
    g46 = dx * dz[1] / (dy / 100. + dy / 140.)
    g45 = dy * dz[1] / (dx / 100. + dx / 120.)
    assert M[4, 4] == pytest.approx(g04 + g45 + g46 + 1e4 * dx * dy, rel=1e-15)


# ---------------------------------------------------------------- SpMV
@pytest.mark.parametrize("dims", TINY)
def test_spmv_unit_vectors_reproduce_columns(dims):
    nx, ny, nz = dims
    A, _, _ = _rand_problem(nx, ny, nz, 4)
    M = A.to_scipy().toarray()
    n = nx * ny * nz
    for i in range(n):
        e = np.zeros(n)
        e[i] = 1.0
        assert np.array_equal(O.spmv(A, e), M[:, i])


def test_spmv_vs_scipy_random():
    A, _, _ = _rand_problem(17, 9, 6, 5)
    x = W.normal01(5, 20, 21, np.arange(A.n))
    y = O.spmv(A, x)
    y2 = A.to_scipy() @ x
    assert np.abs(y - y2).max() <= 1e-14 * np.abs(y2).max()


# ---------------------------------------------------------------- condensed DIA layout
@pytest.mark.parametrize("dims", TINY + [(16, 12, 8)])
def test_dia_layout_closed_forms_and_bruteforce(dims):
    nx, ny, nz = dims
    A, _, _ = _rand_problem(nx, ny, nz, 6)
    n = nx * ny * nz
    vals, ptr, off = O.csr_to_dia(A, nx, ny, nz)
    assert off.tolist() == [0, 1, nx, nx * ny]
    assert ptr.tolist() == [0, n, 2 * n - 1, 3 * n - 1 - nx, 4 * n - 1 - nx - nx * ny]
    M = A.to_scipy().toarray()
    for k in range(4):
        d = np.diagonal(M, offset=int(off[k]))
        assert d.size == n - off[k]
        assert np.array_equal(vals[ptr[k]:ptr[k + 1]], d)
    d1 = vals[ptr[1]:ptr[2]]
    d2 = vals[ptr[2]:ptr[3]]
    d3 = vals[ptr[3]:ptr[4]]
    assert np.count_nonzero(d1 == 0.0) == ny * nz - 1          # x = nx-1 rows
    assert np.count_nonzero(d2 == 0.0) == nx * (nz - 1)        # y = ny-1 rows
    assert np.count_nonzero(d3 == 0.0) == 0
    assert not np.any(np.signbit(vals[vals == 0.0]))           # structural zeros are +0.0


def test_dia_cfg1_element_count():
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    vals, ptr, off = O.csr_to_dia(A, w.nx, w.ny, w.nz)
    assert vals.size == 31711                                   # SURVEY §8 table, cfg 1


def test_alg2_on_dia_equals_csr_spmv():
    # Alg. 2 read 0-based (DESIGN.md R-G1) applied to the extracted diagonals
    nx, ny, nz = 6, 5, 4
    A, _, _ = _rand_problem(nx, ny, nz, 7)
    n = A.n
    vals, ptr, off = O.csr_to_dia(A, nx, ny, nz)
    x = W.normal01(7, 20, 21, np.arange(n))
    y = vals[ptr[0]:ptr[1]] * x
    for k in (1, 2, 3):
        o = int(off[k])
        d = vals[ptr[k]:ptr[k + 1]]
        y[:n - o] += d * x[o:]
        y[o:] += d * x[:n - o]
    ref = O.spmv(A, x)
    assert np.abs(y - ref).max() <= 1e-14 * np.abs(ref).max()


# ---------------------------------------------------------------- solution pins
def test_slab_closed_form_golden():
    gold = np.loadtxt(os.path.join(HERE, "golden", "slab_cfg1.txt"))
    w = W.make_workload(1, n_hot=0)
    A = O.assemble_workload(w)
    r = O.pcg(A, w.power, rtol=1e-9)        # fp64 floor of the true residual here is ~1e-10
    assert r.status == 0
    T = r.x.reshape(w.nz, w.ny, w.nx)
    assert np.abs(T - T[:, :1, :1]).max() < 1e-7               # every column identical
    assert np.abs(T[:, 3, 5] - gold).max() < 1e-7              # golden prints 8 decimals


@pytest.mark.parametrize("dims", TINY + [(9, 8, 6)])
@pytest.mark.parametrize("precond", [0, 1])
def test_pcg_vs_dense_cholesky(dims, precond):
    nx, ny, nz = dims
    A, b, _ = _rand_problem(nx, ny, nz, 8)
    M = A.to_scipy().toarray()
    xs = sla.cho_solve(sla.cho_factor(M), b)
    r = O.pcg(A, b, rtol=1e-10, max_iters=5000, precond=precond)
    assert r.status == 0
    assert np.abs(r.x - xs).max() <= 1e-8 * np.abs(xs).max()
    assert r.iterations <= 2 * A.n + 5   # finite termination, with slack for rounding


def test_pcg_cfg1_vs_dense_cholesky_and_direct():
    w = W.make_workload(1)
    A = O.assemble_workload(w)
    r = O.pcg(A, w.power, rtol=1e-8)
    assert r.status == 0 and r.rel_resid_true <= 1e-8
    assert 200 < r.iterations < 400                             # SURVEY probe: 289
    xs = sla.cho_solve(sla.cho_factor(A.to_scipy().toarray()), w.power)
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    assert np.abs(xd - xs).max() <= 1e-8 * np.abs(xs).max()
    assert np.abs(r.x - xs).max() <= 1e-6 * np.abs(xs).max()
    assert np.all(r.x >= 0)                                     # M-matrix: b >= 0 => x >= 0


def test_pcg_cfg2_vs_direct_solve_and_energy_balance():
    w = W.make_workload(2)
    A = O.assemble_workload(w)
    r = O.pcg(A, w.power, rtol=1e-8)
    assert r.status == 0 and r.rel_resid_true <= 1e-8
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    assert np.abs(r.x - xd).max() <= 1e-6 * np.abs(xd).max()
    top = r.x.reshape(w.nz, -1)[w.nz - 1]
    out = (w.h_top * w.dx * w.dy * top).sum()                   # heat leaving through the top
    assert out == pytest.approx(w.power.sum(), rel=1e-6)


def test_transient_step_vs_direct_and_energy_balance():
    w = W.make_workload(5, nx=48, ny=40, nz=16, n_hot=8)
    A = O.assemble_workload(w)
    T = np.zeros(w.n)
    cap = np.repeat(w.cvol * w.dx * w.dy * w.dz / w.dt, w.nx * w.ny)
    for step in (1, 2, 3):
        P = W.power_for_step(w, step)
        b = O.transient_rhs(w, P, T)
        assert np.allclose(b, P + cap * T, rtol=1e-15, atol=0)
        r = O.pcg(A, b, x0=T, rtol=1e-10)
        assert r.status == 0
        xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, b, w.cvol, w.dt)
        assert np.abs(r.x - xd).max() <= 1e-7 * max(np.abs(xd).max(), 1e-30)
        top = r.x.reshape(w.nz, -1)[w.nz - 1]
        lhs = (cap * (r.x - T)).sum() + (w.h_top * w.dx * w.dy * top).sum()
        assert lhs == pytest.approx(P.sum(), rel=1e-7)          # eq. (5) summed over cells
        T = r.x


def test_paperlike_anisotropic_stack_vs_direct_solve():
    # cfg 6: the paper's layer thicknesses 2-1000 um with 50 um cells: diagonals differ by 1e5
    w = W.make_workload(6, nx=40, ny=36, nz=10, n_hot=6)
    A = O.assemble_workload(w)
    r = O.pcg(A, w.power, rtol=1e-9)
    assert r.status == 0
    xd = solve_layered(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.kappa_layer, w.h_top, w.power)
    assert np.abs(r.x - xd).max() <= 1e-7 * np.abs(xd).max()
    top = r.x.reshape(w.nz, -1)[w.nz - 1]
    assert (w.h_top * w.dx * w.dy * top).sum() == pytest.approx(w.power.sum(), rel=1e-7)


def test_pcg_lognormal_small_vs_cholesky():
    w = W.make_workload(3, nx=12, ny=10, nz=16, n_hot=6)
    A = O.assemble_workload(w)
    xs = sla.cho_solve(sla.cho_factor(A.to_scipy().toarray()), w.power)
    r = O.pcg(A, w.power, rtol=1e-10)
    assert r.status == 0
    assert np.abs(r.x - xs).max() <= 1e-7 * np.abs(xs).max()


# ---------------------------------------------------------------- properties of the iteration
def test_cg_anorm_error_monotone_and_precond_agree():
    A, b, _ = _rand_problem(6, 5, 4, 9)
    M = A.to_scipy().toarray()
    xs = sla.cho_solve(sla.cho_factor(M), b)
    prev = None
    for k in range(0, 40, 3):
        x = O.pcg_window(A, b, np.zeros(A.n), k)
        e = x - xs
        en = float(e @ (M @ e))
        if prev is not None:
            assert en <= prev * (1 + 1e-9)
        prev = en
    x0 = O.pcg(A, b, rtol=1e-10, max_iters=5000, precond=0).x
    x1 = O.pcg(A, b, rtol=1e-10, max_iters=5000, precond=1).x
    assert np.abs(x0 - x1).max() <= 1e-9 * np.abs(xs).max()


def test_zero_rhs_and_warm_start():
    A, b, _ = _rand_problem(5, 4, 3, 10)
    r = O.pcg(A, np.zeros(A.n), x0=np.ones(A.n))
    assert r.status == 0 and r.iterations == 0 and np.all(r.x == 0)
    xs = O.pcg(A, b, rtol=1e-10, max_iters=5000).x
    r2 = O.pcg(A, b, x0=xs, rtol=1e-8)
    assert r2.iterations == 0 and np.array_equal(r2.x, xs)
