"""Helpers for the -m gpu parity tests: workload -> C-ABI objects (through the Python binding)."""
import numpy as np


def grid_from_workload(w, device="cuda"):
    import torch
    import paper_2606_17850_b200 as cu
    kap = w.kappa_cell if w.kappa_cell is not None else w.kappa_layer
    kt = torch.from_numpy(np.ascontiguousarray(kap)).to(device)
    return cu.Grid(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, kt, w.h_top, w.cvol, w.dt)


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def gpu_solve(w, b, precision, x0=None, rtol=1e-8, max_iters=200000, period=None, precond=1):
    """Build + solve through the C ABI; returns (x numpy, Result, DiaMatrix, Solver)."""
    import torch
    import paper_2606_17850_b200 as cu
    g = grid_from_workload(w)
    A = cu.DiaMatrix(g)
    opts = cu.Opts(precision=precision, rtol=rtol, max_iters=max_iters,
                   true_resid_period=period or w.true_resid_period, preconditioner=precond)
    S = cu.Solver(A, opts)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda") if x0 is None else to_dev(x0)
    S.solve(to_dev(b), x)
    res = S.result()
    return x.cpu().numpy(), res, A, S
