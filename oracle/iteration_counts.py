"""Writes tests/golden/oracle_iterations.txt: how many Alg.-1 iterations (M = diag A, rtol of the
workload, verified on the true residual: SURVEY.md §8(c) C4) the CPU ORACLE needs on the BASELINE workloads it can
solve in minutes.  TEST INFRASTRUCTURE: calls only oracle/ and the seeded input generators (workloads/); nothing
from the CUDA path.  bench.py's reference arm multiplies its measured seconds per oracle iteration by these counts
(the oracle's own, not the GPU's).

  python -m oracle.iteration_counts [cfg ...]        # default: 1 2 6 3   (cfg 3: several minutes on 8 cores)
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402
from oracle import oracle as O  # noqa: E402

OUT = os.path.join(ROOT, "tests", "golden", "oracle_iterations.txt")
HEADER = """# Iterations of the CPU oracle's Jacobi-PCG (oracle_pcg: Alg. 1, PAPER.md:145-168, M = diag A, stop on a verified true
# residual <= rtol ||b||, SURVEY.md §8(c) C4) on the full-size BASELINE workloads, written by oracle/iteration_counts.py
# (calls only oracle/ and workloads/).  Columns: cfg  N  rtol  iterations  true_rel_resid  seconds  threads
"""


def main(cfgs):
    rows = {}
    if os.path.exists(OUT):
        for line in open(OUT):
            if line.strip() and not line.startswith("#"):
                rows[int(line.split()[0])] = line.rstrip("\n")
    for cfg in cfgs:
        w = W.make_workload(cfg)
        A = O.assemble_workload(w)
        b = w.power if not w.transient else O.transient_rhs(w, w.power, np.zeros(w.n))
        t0 = time.time()
        res = O.pcg(A, b, rtol=w.rtol)
        dt = time.time() - t0
        assert res.status == 0
        rows[cfg] = f"{cfg} {w.n} {w.rtol:g} {res.iterations} {res.rel_resid_true:.6e} {dt:.1f} {O.num_threads()}"
        print(rows[cfg], flush=True)
        with open(OUT, "w") as f:
            f.write(HEADER)
            for k in sorted(rows):
                f.write(rows[k] + "\n")


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [1, 2, 6, 3])
