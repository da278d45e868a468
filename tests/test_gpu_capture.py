"""include/cuth.h: "every call is asynchronous on `stream` and never synchronises" -- checked the hard way: the calls
that do not launch a graph themselves are recorded under CUDA STREAM CAPTURE (a call that synchronised, or that made a
pageable cudaMemcpyAsync as round 1's cuth_build_dia did, would invalidate the capture), and the captured graph replays
to the same bits as the eager calls.  cuth_pcg_solve launches its own CUDA graph and is therefore enqueued outside."""
import numpy as np
import pytest

import workloads as W
from gpu_util import grid_from_workload, to_dev

pytestmark = pytest.mark.gpu


def test_build_spmv_and_noalloc_residual_are_capturable():
    import torch
    import paper_2606_17850_b200 as cu
    w = W.make_workload(3, nx=40, ny=24, nz=6, n_hot=4)
    g = grid_from_workload(w)
    x = to_dev(W.normal01(w.seed, 80, 81, np.arange(w.n)) + 2.0)
    b = to_dev(w.power)
    # eager reference
    buf0 = torch.zeros(cu.cuth_dia_bytes(g), dtype=torch.uint8, device="cuda")
    cu.cuth_build_dia(g, buf0)
    y0 = torch.empty_like(x); y1 = torch.empty_like(x); t0 = torch.empty_like(x); o0 = torch.zeros(4, dtype=torch.float64, device="cuda")
    cu.cuth_spmv(buf0, g, cu.FP64, x, y0)
    cu.cuth_spmv(buf0, g, cu.MIXED, x, y1)
    cu.cuth_residual_noalloc(buf0, g, b, x, o0, t=t0)
    torch.cuda.synchronize()
    # the same calls under capture, into fresh buffers
    buf = torch.zeros_like(buf0)
    z0 = torch.zeros_like(x); z1 = torch.zeros_like(x); t1 = torch.zeros_like(x); o1 = torch.zeros(4, dtype=torch.float64, device="cuda")
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        cu.cuth_build_dia(g, buf)
        cu.cuth_spmv(buf, g, cu.FP64, x, z0)
        cu.cuth_spmv(buf, g, cu.MIXED, x, z1)
        cu.cuth_residual_noalloc(buf, g, b, x, o1, t=t1)
    torch.cuda.synchronize()
    assert not bool(z0.any()) and not bool(buf.any())            # nothing ran during capture
    for _ in range(2):                                           # replay twice
        graph.replay()
        torch.cuda.synchronize()
        assert bool((buf == buf0).all())                         # the matrix object, byte for byte
        for a, r in ((z0, y0), (z1, y1), (t1, t0), (o1, o0)):
            assert np.array_equal(a.cpu().numpy().view(np.uint64), r.cpu().numpy().view(np.uint64))
        z0.zero_(); z1.zero_(); t1.zero_(); o1.zero_(); buf.zero_()
