"""No-GPU checks of the C-ABI boundary: the library loads, exports every symbol include/cuth.h
declares, and its pure-host entry points (sizes, layout view, argument errors) behave."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cu():
    from paper_2606_17850_b200 import build
    build.build()
    import paper_2606_17850_b200 as cu
    return cu


def test_exports_match_header(cu):
    hdr = open(os.path.join(ROOT, "include", "cuth.h")).read()
    declared = set(re.findall(r"\b(cuth_[a-z0-9_]+)\s*\(", hdr))
    declared -= {"cuth_status_t"}
    lib = cu.load_library()
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(cu.exported_symbols())
    # SURVEY.md §8(b) "no global state": the library has no process-wide setter; kernel variants are per call
    assert not [n for n in declared if n.startswith("cuth_set_")]
    assert "cuth_tuning_t tuning;" in hdr


def test_struct_sizes_match_the_header(cu):
    """The ctypes mirrors of the ABI structs have the sizes the C compiler gives them (a quick layout check:
    gcc on the header itself)."""
    import subprocess
    import tempfile
    from paper_2606_17850_b200 import binding as B
    src = '#include <stdio.h>\n#include "cuth.h"\nint main(){printf("%zu %zu %zu %zu %zu\\n", sizeof(cuth_grid_t), ' \
          'sizeof(cuth_opts_t), sizeof(cuth_result_t), sizeof(cuth_tuning_t), sizeof(cuth_import_report_t));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "t.c"), "w").write(src)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), os.path.join(d, "t.c"), "-o", os.path.join(d, "t")],
                       check=True)
        out = subprocess.run([os.path.join(d, "t")], check=True, capture_output=True, text=True).stdout.split()
    want = [C.sizeof(B.cuth_grid_t), C.sizeof(B.cuth_opts_t), C.sizeof(B.cuth_result_t), C.sizeof(B.cuth_tuning_t),
            C.sizeof(B.cuth_import_report_t)]
    assert [int(v) for v in out] == want


def test_bad_tuning_and_precision_values_are_argument_errors(cu):
    g = cu.Grid(8, 8, 4, 1e-6, 1e-6, np.full(4, 1e-6), None, 1e4)
    lib = cu.load_library()
    p = C.c_void_p(4096)
    for kw in (dict(traversal=3), dict(loop_mode=5), dict(k1_variant=4), dict(cheb_fusion=4), dict(pair_rows=12),
               dict(pair_occupancy=1)):
        o = cu.Opts(tuning=cu.Tuning(**kw))
        assert lib.cuth_pcg_solve(p, g.ref(), C.byref(o), p, p, p, 1 << 30, p, None) == -3, kw
        t = cu.Tuning(**kw)
        assert lib.cuth_spmv_tuned(p, g.ref(), 0, C.byref(t), p, C.c_void_p(8192), None) == -3, kw
    o = cu.Opts(precision=9)
    assert lib.cuth_pcg_solve(p, g.ref(), C.byref(o), p, p, p, 1 << 30, p, None) == -3
    o = cu.Opts(precision=cu.MIXED_STD32, preconditioner=cu.PRECOND_CHEBYSHEV, cheb_lmin=1.0, cheb_lmax=2.0)
    assert lib.cuth_pcg_solve(p, g.ref(), C.byref(o), p, p, p, 1 << 30, p, None) == -3      # ablation: Jacobi / none only


def test_layout_closed_forms_host_side(cu):
    for nx, ny, nz in [(4, 3, 2), (32, 32, 8), (256, 256, 16), (4096, 4096, 8)]:
        g = cu.Grid(nx, ny, nz, 1e-6, 1e-6, np.full(nz, 1e-6), None, 1e4)
        n = nx * ny * nz
        lib = cu.load_library()
        ptr = (C.c_int64 * 5)()
        off = (C.c_int64 * 4)()
        rc = lib.cuth_dia_view(C.c_void_p(4096), g.ref(), None, None, None, ptr, off)
        assert rc == 0
        assert list(off) == [0, 1, nx, nx * ny]
        assert list(ptr) == [0, n, 2 * n - 1, 3 * n - 1 - nx, 4 * n - 1 - nx - nx * ny]
        e = ptr[4]
        assert cu.cuth_dia_bytes(g) >= 8 * e + 4 * e + 8 * n
        assert cu.cuth_workspace_bytes(g, cu.Opts()) >= 3 * 8 * n


def test_degenerate_dims_rejected(cu):
    for dims in [(1, 4, 4), (4, 1, 4), (4, 4, 1), (0, 4, 4)]:
        g = cu.Grid(*dims, 1e-6, 1e-6, np.full(max(dims[2], 1), 1e-6), None, 1e4)
        assert cu.cuth_dia_bytes(g) == 0
        lib = cu.load_library()
        assert lib.cuth_build_dia(g.ref(), C.c_void_p(4096), 1 << 20, None) == -2   # CUTH_ERR_DIMS
    g = cu.Grid(4, 4, 4, 1e-6, 1e-6, np.full(4, 1e-6), None, 1e4)
    lib = cu.load_library()
    assert lib.cuth_build_dia(g.ref(), None, 1 << 20, None) == -1                   # NULL
    assert lib.cuth_spmv(C.c_void_p(4096), g.ref(), 7, C.c_void_p(4096), C.c_void_p(8192), None) == -3
    assert lib.cuth_spmv(C.c_void_p(4096), g.ref(), 0, C.c_void_p(4100), C.c_void_p(8192), None) == -5


def test_no_cpu_fallback_without_device(cu):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    g = cu.Grid(4, 4, 4, 1e-6, 1e-6, np.full(4, 1e-6), None, 1e4)
    with pytest.raises(RuntimeError):
        cu.DiaMatrix(g)


def test_tridiag_extremes_vs_lapack(cu):
    """Host half of the Lanczos setup (Sturm bisection) against LAPACK on random and on Lanczos tridiagonals."""
    import scipy.linalg as sla
    import workloads as W
    for m, seed in ((1, 1), (2, 2), (7, 3), (40, 4), (120, 5)):
        a = 1e-3 * (1.0 + W.uniform01(seed, 60, np.arange(m)))
        b = 5e-4 * W.uniform01(seed, 61, np.arange(max(m - 1, 1)))
        lo, hi = cu.cuth_tridiag_extremes(a, b[:max(m - 1, 0)] if m > 1 else np.zeros(1))
        w = sla.eigvalsh_tridiagonal(a, b[:m - 1]) if m > 1 else a
        assert lo == pytest.approx(w[0], rel=1e-12, abs=1e-18) and hi == pytest.approx(w[-1], rel=1e-12)
    from oracle import oracle as O
    wl = W.make_workload(1)
    A = O.assemble_workload(wl)
    al, be = O.lanczos(A, wl.power, 30)
    lo, hi = cu.cuth_tridiag_extremes(al, be[:len(al) - 1])
    lo_o, hi_o = O.ritz_extremes(al, be)
    assert lo == pytest.approx(lo_o, rel=1e-9) and hi == pytest.approx(hi_o, rel=1e-12)


def test_layout_golden_sizes(cu):
    """ptr[] of the C ABI against the element counts tabulated for the five BASELINE grids (tests/golden)."""
    rows = np.loadtxt(os.path.join(ROOT, "tests", "golden", "layout_sizes.txt"), dtype=np.int64)
    lib = cu.load_library()
    for cfg, nx, ny, nz, n, e in rows:
        g = cu.Grid(int(nx), int(ny), int(nz), 1e-6, 1e-6, np.full(int(nz), 1e-6), None, 1e4)
        ptr = (C.c_int64 * 5)()
        off = (C.c_int64 * 4)()
        assert lib.cuth_dia_view(C.c_void_p(4096), g.ref(), None, None, None, ptr, off) == 0
        assert nx * ny * nz == n and ptr[4] == e and ptr[1] == n


def test_cheb_launch_schedule_host_side(cu):
    """cuth_cheb_launches (pure host): k - 1 launches with one pass per kernel (R-C3: the dead k-th SpMV of
    Alg. 3 is skipped); with two passes per kernel the k - 3 middle passes pair up, FIRST and LAST stay -- and
    where the TMA kernel is available (nx % 4 == 0 and a driver that can encode tensor maps) an odd middle pass
    left over shares its launch with LAST."""
    dz = np.full(16, 1e-6)
    big = cu.Grid(1024, 1024, 16, 1e-6, 1e-6, dz, None, 1e4)           # nx % 4 == 0
    even = cu.Grid(34, 32, 16, 1e-6, 1e-6, dz, None, 1e4)              # even nx, not a multiple of 4: no TMA
    odd = cu.Grid(1023, 1024, 16, 1e-6, 1e-6, dz, None, 1e4)           # odd nx: never pairs
    mk = lambda prec, k, mode: cu.Opts(prec, 1e-8, 1000, 20, cu.PRECOND_CHEBYSHEV, k, 1e-3, 1.0, cu.CHEB_DEFAULT,
                                       cu.Tuning(cheb_fusion=mode))
    for k in (3, 4, 5, 30, 31):
        mids = k - 3
        plain = (2 + mids // 2 + mids % 2, mids // 2)              # FIRST, pairs, odd MID, LAST
        fused = (2 + mids // 2, mids // 2 + mids % 2) if mids % 2 else plain   # odd MID + LAST in one launch
        assert cu.cuth_cheb_launches(big, mk(cu.MIXED, k, 1)) == (k - 1, 0)
        for mode in (0, 2):
            assert cu.cuth_cheb_launches(big, mk(cu.MIXED, k, mode)) in (plain, fused)
            assert cu.cuth_cheb_launches(even, mk(cu.MIXED, k, mode)) == plain
            assert cu.cuth_cheb_launches(odd, mk(cu.MIXED, k, mode)) == (k - 1, 0)
            assert cu.cuth_cheb_launches(big, mk(cu.FP64, k, mode)) == (k - 1, 0)          # fp64 apply: single passes
        assert cu.cuth_cheb_launches(big, mk(cu.MIXED, k, 3)) == plain                      # never the TMA kernel
    assert cu.cuth_cheb_launches(big, cu.Opts(cu.MIXED, 1e-8, 1000, 20)) == (0, 0)   # Jacobi: no apply


def test_kernel_choice_queries_host_side(cu):
    """cuth_traversal / cuth_loop_home / cuth_launches_per_iteration (pure host) on the BASELINE grids: the rules stated in
    include/cuth.h (cuth_tuning_t).  Where the driver cannot encode tensor maps (this CPU box) the TMA-dependent choices
    fall back, and without a device there is no cooperative launch: hence the sets."""
    mk = lambda nx, ny, nz: cu.Grid(nx, ny, nz, 1e-6, 1e-6, np.full(nz, 1e-6), None, 1e4)
    o64, omx = cu.Opts(cu.FP64), cu.Opts(cu.MIXED)
    cfg1, cfg2, cfg3, cfg4, cfg5 = mk(32, 32, 8), mk(256, 256, 16), mk(1024, 1024, 16), mk(4096, 4096, 8), mk(512, 512, 16)
    # cfg 1 fits one thread-block cluster; cfg 2 is flat in one persistent kernel; cfg 3 / 4 z-march in the graph
    assert (cu.cuth_traversal(cfg1, omx), cu.cuth_loop_home(cfg1, omx), cu.cuth_launches_per_iteration(cfg1, omx)) == (1, 3, 0)
    # (without a device there is no cooperative launch: the graph loop with its three flat kernels)
    assert (cu.cuth_traversal(cfg2, omx), cu.cuth_loop_home(cfg2, omx), cu.cuth_launches_per_iteration(cfg2, omx)) in ((1, 2, 0), (1, 1, 3))
    for g in (cfg3, cfg4):
        for o in (o64, omx):
            assert (cu.cuth_traversal(g, o), cu.cuth_loop_home(g, o)) == (2, 1)
    assert cu.cuth_launches_per_iteration(cfg3, omx) == 2 and cu.cuth_launches_per_iteration(cfg4, o64) == 2
    assert cu.cuth_launches_per_iteration(cfg4, omx) in (2, 3)          # 3 = thin stack: TMA K1 early + LDG K1 late
    assert cu.cuth_loop_home(cfg5, omx) in (1, 2)                       # graph with the TMA K1, else the persistent kernel
    # forced variants
    assert cu.cuth_traversal(cfg3, cu.Opts(cu.FP64, tuning=cu.Tuning(traversal=1))) == 1
    assert cu.cuth_traversal(cfg2, cu.Opts(cu.FP64, tuning=cu.Tuning(traversal=2))) == 2
    assert cu.cuth_loop_home(cfg1, cu.Opts(cu.FP64, tuning=cu.Tuning(loop_mode=4))) == 3
    assert cu.cuth_loop_home(cfg1, cu.Opts(cu.FP64, tuning=cu.Tuning(loop_mode=2))) in (2, 1)
    assert cu.cuth_loop_home(cfg1, cu.Opts(cu.FP64, tuning=cu.Tuning(loop_mode=1))) == 1
    assert cu.cuth_launches_per_iteration(cfg4, cu.Opts(cu.MIXED, tuning=cu.Tuning(k1_variant=2))) == 2
    assert cu.cuth_traversal(cfg3, cu.Opts(cu.MIXED_STD32)) == 1          # the ablation operator exists in the flat traversal only


def test_batch_and_import_host_side(cu):
    """Pure-host behaviour of the two calls added last: batch workspace size (0 on a bad count, grows by three
    vectors per right-hand side) and the argument checks that come before any CUDA call."""
    g = cu.Grid(32, 32, 8, 1e-6, 1e-6, np.full(8, 1e-6), None, 1e4)
    n = 32 * 32 * 8
    assert cu.cuth_batch_workspace_bytes(g, 0) == 0 and cu.cuth_batch_workspace_bytes(g, 33) == 0
    sizes = [cu.cuth_batch_workspace_bytes(g, k) for k in range(1, 33)]
    assert all(b - a == 3 * 8 * n for a, b in zip(sizes, sizes[1:]))            # r, p, mu per right-hand side
    assert sizes[0] >= 3 * 8 * n and sizes[0] % 256 == 0
    lib = cu.load_library()
    from paper_2606_17850_b200.binding import cuth_import_report_t
    rep = cuth_import_report_t()
    p = C.c_void_p(4096)
    big = cu.cuth_dia_bytes(g)
    assert lib.cuth_import_csr(g.ref(), None, p, p, None, p, big, C.byref(rep), None) == -1       # NULL rowptr
    assert lib.cuth_import_csr(g.ref(), p, p, p, None, None, big, C.byref(rep), None) == -1       # NULL matrix
    assert lib.cuth_import_csr(g.ref(), p, p, p, None, p, big - 1, C.byref(rep), None) == -4      # buffer too small
    assert lib.cuth_import_csr(g.ref(), C.c_void_p(4100), p, p, None, p, big, C.byref(rep), None) == -5
    neg = np.full(8, -1.0)
    assert lib.cuth_import_csr(g.ref(), p, p, p, neg.ctypes.data_as(C.c_void_p), p, big, C.byref(rep), None) == -3
    assert lib.cuth_import_coo(g.ref(), None, p, p, C.c_int64(10), None, p, big, C.byref(rep), None) == -1
    assert lib.cuth_import_coo(g.ref(), p, p, p, C.c_int64(-1), None, p, big, C.byref(rep), None) == -3
    assert lib.cuth_import_coo(g.ref(), p, p, p, C.c_int64(10), None, p, big - 1, C.byref(rep), None) == -4
    bad = cu.Grid(1, 4, 4, 1e-6, 1e-6, np.full(4, 1e-6), None, 1e4)
    assert lib.cuth_import_csr(bad.ref(), p, p, p, None, p, big, C.byref(rep), None) == -2
    o = cu.Opts()
    assert lib.cuth_pcg_solve_batch(p, g.ref(), C.byref(o), 0, p, p, p, 1 << 30, p, None) == -3   # nrhs out of range
    assert lib.cuth_pcg_solve_batch(p, g.ref(), C.byref(o), 33, p, p, p, 1 << 30, p, None) == -3
    oc = cu.Opts(preconditioner=cu.PRECOND_CHEBYSHEV, cheb_lmin=1.0, cheb_lmax=2.0)
    assert lib.cuth_pcg_solve_batch(p, g.ref(), C.byref(oc), 2, p, p, p, 1 << 30, p, None) == -3  # no Chebyshev batch
    assert lib.cuth_pcg_solve_batch(p, g.ref(), C.byref(o), 2, None, p, p, 1 << 30, p, None) == -1
    assert lib.cuth_pcg_solve_batch(p, g.ref(), C.byref(o), 2, p, p, p, 1024, p, None) == -4      # workspace too small
