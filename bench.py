#!/usr/bin/env python
"""bench.py -- PCG time-to-solution and HBM roofline of the cuth hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--precision fp64|mixed]
  python bench.py --impl reference ...        # the CPU oracle on the host cores, bounded sample

One "step" = one whole solve of the workload (cuth_pcg_solve to a verified true relative residual
<= 1e-8; for config 5: the whole 200-step backward-Euler trace) on synthetic seeded inputs (workloads/).  The default
workload is BASELINE.json configs[2] (1024x1024x16, 16.8 M unknowns): the first of the two grids the
metric's HBM target is quoted on, and the largest whose full solve keeps the default run within
minutes.  N > 1: independent replicas, one per GPU ("replicas only", no collective on
the data path); the time is the max over ranks.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum per launch from `ncu --set full` captures of the dominant
# kernel (profiles/r1e_cfg3_fp64_k1x2.md, r1d, r1c); null for workloads/kernels not captured.
NCU_TRAFFIC_BYTES = {("cfg3_steady_1024x1024x16_lognormal", "k_fused_pspmv", "fp64"): 1.3200e9,   # profiles/r2d_cfg3_mixed_final.md (TMA-staged K1)
                     ("cfg3_steady_1024x1024x16_lognormal", "k_fused_pspmv", "mixed"): 1.0412e9,  # profiles/r2d_cfg3_mixed_final.md (fp32-stored operator)
                     ("cfg3_steady_1024x1024x16_lognormal", "k_cheb_pair", "mixed"): 518.3e6,    # profiles/r1i_cfg3_default_and_cheb16.md
                     ("cfg4_steady_4096x4096x8", "k_cheb_pair", "mixed"): 4.477e9,                 # profiles/r1h_cheb_pair_tma.md
                     ("cfg4_steady_4096x4096x8", "k_fused_pspmv", "fp64"): 10.786e9,               # profiles/r1j_cfg4_fp64_k1.md
                     }

METRIC = "pcg_time_to_solution"
UNIT = "s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def m_ratio(w):
    return (4 * w.n - 1 - w.nx - w.nx * w.ny) / w.n


def bytes_per_row(w, what):
    """Algorithmic bytes per matrix row."""
    m = m_ratio(w)
    # the fused K1 takes M = diag A from the D0 its SpMV reads (fp64 operator), so a fused fp64 iteration
    # moves 8m + 80, not the 8m + 88 of the three-kernel path (which reads 1/D0 in k_pupdate)
    return {"spmv_fp64": 8 * m + 16, "spmv_mixed": 4 * (m - 1) + 16,
            "iter_fp64": 8 * m + 88, "iter_fp64_fused": 8 * m + 80, "iter_mixed": 4 * (m - 1) + 88,
            # fused path, early stage: 1/D0 is read as fp32 in K1 and in K2 (4 + 4 B instead of 8 + 8)
            "iter_mixed_fused": 4 * (m - 1) + 80}[what]


def max_over_ranks(value_ms: float, world: int, device="cpu") -> float:
    """Replicas-only multi-GPU timing: every rank times its own solve, the job's time is the MAX over
    ranks (no data-path collective; this all_reduce of one float is measurement plumbing only)."""
    if world <= 1:
        return float(value_ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value_ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown," \
        "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown," \
        "clocks_event_reasons.sw_power_cap"

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [t.strip() for t in line.split(",")]
            if len(c) < 8:
                continue
            try:
                sm.append(float(c[0]))
                mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm))
        return out


# Iterations to convergence used when a measured seconds-per-iteration of the oracle is turned into a time to solution.
# cfg 1, 2, 3, 6: the ORACLE's own count (tests/golden/oracle_iterations.txt, written by oracle/iteration_counts.py).
# cfg 4, 5: a full oracle solve takes hours; the count below is the FP64 GPU solve's and
# the result is labelled "extrapolated with the GPU's iteration count".
GPU_FP64_ITERS = {4: 9791, 5: 115916}


def oracle_iterations(cfg):
    path = os.path.join(ROOT, "tests", "golden", "oracle_iterations.txt")
    if os.path.exists(path):
        for line in open(path):
            if line.strip() and not line.startswith("#") and int(line.split()[0]) == cfg:
                return int(line.split()[3]), "the oracle's own iteration count (tests/golden/oracle_iterations.txt)"
    if cfg in GPU_FP64_ITERS:
        return GPU_FP64_ITERS[cfg], "the FP64 GPU solve's iteration count (a full oracle solve takes hours)"
    return None, ""


WIN_SHORT, WIN_LONG = 20, 91          # oracle timing windows: seconds per iteration = (t_long - t_short) / 71


def oracle_s_per_iteration(O, A, b, n):
    """Seconds per Alg.-1 iteration of the oracle as it stands, from TWO windows of 20 and 91 iterations: the
    difference cancels what each oracle_pcg_window call does besides iterating (it allocates and zero-fills five
    vectors and forms r0), so the same number comes out of both bench arms whatever the window length."""
    x0 = np.zeros(n)
    t0 = time.time()
    O.pcg_window(A, b, x0, WIN_SHORT)
    t1 = time.time()
    O.pcg_window(A, b, x0, WIN_LONG)
    t2 = time.time()
    return ((t2 - t1) - (t1 - t0)) / (WIN_LONG - WIN_SHORT), t2 - t0


def cpu_oracle_baseline(w, cfg, x_gpu=None, full=None, out=None):
    """The oracle as it stands on the host cores.  cfg 1, 2, 3, 6 (`full`): ONE solve to convergence, measured --
    time to solution, iterations, and max |x_gpu - x_oracle| at full size.  cfg 4, 5: seconds per iteration from the
    two windows, times the iteration count (extrapolated, labelled)."""
    from oracle import oracle as O
    t0 = time.time()
    A = O.assemble_workload(w)
    t_asm = time.time() - t0
    b = w.power if not w.transient else O.transient_rhs(w, w.power, np.zeros(w.n))
    if out is not None:
        out["A"], out["b"] = A, b
    if full is None:
        full = cfg in (1, 2, 3, 6)
    s_it, t_win = oracle_s_per_iteration(O, A, b, w.n)
    base = {"unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "s_per_iteration": s_it, "assembly_s": t_asm}
    if full:
        t0 = time.time()
        ref = O.pcg(A, b, rtol=w.rtol)
        dt = time.time() - t0
        base.update(value=dt, iterations=ref.iterations, rel_resid_true=ref.rel_resid_true,
                    sample=f"ONE full solve of {w.name} by the CSR fp64 oracle to a verified true residual <= {w.rtol:g}: "
                           f"{ref.iterations} iterations in {dt:.1f} s (measured, not extrapolated); windows of {WIN_SHORT} / "
                           f"{WIN_LONG} iterations give {s_it * 1e3:.2f} ms/iteration; CSR assembly {t_asm:.1f} s not included")
        if x_gpu is not None:
            base["max_abs_diff_gpu_vs_oracle_K"] = float(np.abs(x_gpu - ref.x).max())
            base["max_rel_diff_gpu_vs_oracle"] = float(np.abs(x_gpu - ref.x).max() / np.abs(ref.x).max())
    else:
        its, src = oracle_iterations(cfg)
        base.update(value=s_it * its, iterations=its,
                    sample=f"windows of {WIN_SHORT} and {WIN_LONG} Alg.-1 iterations of the CSR fp64 oracle on {w.name} ({t_win:.1f} s): "
                           f"{s_it * 1e3:.2f} ms/iteration, EXTRAPOLATED to {its} iterations = {src}; CSR assembly "
                           f"{t_asm:.1f} s not included")
    return base


def run_reference(args):
    """--impl reference: the oracle on the host cores.  Each step = the two timing windows (20 + 91 iterations) of the
    same workload; value = seconds per iteration x iterations to convergence (the oracle's own count where a golden
    one exists).  The GPU arm's cpu_baseline runs the full solve once and reports the measured time beside it."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = W.make_workload(args.config)
    from oracle import oracle as O
    A = O.assemble_workload(w)
    b = w.power if not w.transient else O.transient_rhs(w, w.power, np.zeros(w.n))
    its, src = oracle_iterations(args.config)
    for _ in range(args.warmup):
        O.pcg_window(A, b, np.zeros(w.n), 2)
    s_its, t0 = [], time.time()
    for _ in range(args.steps):
        s_it, _ = oracle_s_per_iteration(O, A, b, w.n)
        s_its.append(s_it)
    dt = (time.time() - t0) / args.steps
    s_it = float(np.median(s_its))
    val = s_it * its
    sample = (f"each step = windows of {WIN_SHORT} and {WIN_LONG} Alg.-1 iterations of the CSR fp64 oracle on {w.name}; "
              f"median {s_it * 1e3:.2f} ms/iteration over {args.steps} steps, times {its} iterations = {src}")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_unknowns": w.n, "grid": [w.nx, w.ny, w.nz], "rtol": w.rtol,
                       "preconditioner": "jacobi", "precision": "fp64", "parallelism": "host cores"},
            "iterations": its, "s_per_iteration": s_it,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_batch(args):
    """`--batch NRHS`: cuth_pcg_solve_batch on NRHS seeded power maps of the workload (FP64, Jacobi) against the same
    NRHS systems solved one after the other with cuth_pcg_solve.  One step = the whole batch."""
    import torch
    import paper_2606_17850_b200 as cu
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    w = W.make_workload(args.config)
    nrhs = args.batch
    kap = w.kappa_cell if w.kappa_cell is not None else w.kappa_layer
    g = cu.Grid(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, torch.from_numpy(np.ascontiguousarray(kap)).cuda(), w.h_top)
    A = cu.DiaMatrix(g)
    mixed = args.precision == "mixed"
    opts = cu.Opts(precision=cu.MIXED if mixed else cu.FP64, rtol=w.rtol, max_iters=200000,
                   true_resid_period=w.true_resid_period)
    idx = np.arange(w.n)
    B = np.stack([w.power * (0.25 + 1.5 * W.uniform01(w.seed, 100 + s, idx)) if s else w.power for s in range(nrhs)])
    b_host = torch.from_numpy(B).pin_memory()
    x_host = torch.empty_like(b_host).pin_memory()
    b = b_host.cuda()
    b_stage = torch.empty_like(b)
    x = torch.zeros_like(b)
    SB = cu.BatchSolver(A, nrhs, opts)
    S1 = cu.Solver(A, opts)
    stream = torch.cuda.current_stream()

    def batch_pass(from_host):
        x.zero_()
        if from_host:
            b_stage.copy_(b_host, non_blocking=True)
        SB.solve(b_stage if from_host else b, x)
        if from_host:
            x_host.copy_(x, non_blocking=True)

    def seq_pass():
        x.zero_()
        for s in range(nrhs):
            S1.solve(b[s], x[s])

    def timed(fn, *a):
        for _ in range(args.warmup):
            fn(*a)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for e0, e1 in ev:
            e0.record(stream)
            fn(*a)
            e1.record(stream)
        torch.cuda.synchronize()
        return float(np.mean([e0.elapsed_time(e1) for e0, e1 in ev]))

    sampler = ClockSampler(0)
    ms_batch = timed(batch_pass, False)
    clocks = sampler.stop()
    res = SB.results()
    xb = x.cpu().numpy().copy()
    ms_e2e = timed(batch_pass, True)
    ms_seq = timed(seq_pass)
    xs = x.cpu().numpy()
    its = [r.iterations for r in res]
    peak, peak_src = peaks()
    m = m_ratio(w)
    # three phases per iteration: (8m + 8)/S matrix and 1/D0 bytes shared by S = 4 right-hand sides,
    # 88 vector bytes per right-hand side
    bytes_it = sum(its) * (88 + (8 * m + 16) / min(4, nrhs)) * w.n
    line = {"metric": METRIC, "value": ms_batch * 1e-3, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_batch, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_unknowns": w.n, "grid": [w.nx, w.ny, w.nz],
                       "precision": "mixed" if mixed else "fp64",
                       "preconditioner": "jacobi", "rtol": w.rtol, "batch_nrhs": nrhs,
                       "l2_policy": "batched small-grid case: the working set of all right-hand sides is what it is; no flush",
                       "parallelism": "1 GPU"},
            "iterations": its, "status": [r.status_name for r in res],
            "max_rel_resid_true": max(r.rel_resid_true for r in res),
            "solves_per_s": nrhs / (ms_batch * 1e-3),
            "sequential_single_solves_ms": ms_seq, "speedup_vs_sequential": ms_seq / ms_batch,
            "max_rel_diff_vs_single_solves": float(np.abs(xb - xs).max() / np.abs(xs).max()),
            "roofline": {"bound": "hbm", "kernel": "k_pcg_batch (whole solve, persistent)",
                         "achieved": bytes_it / ms_batch / 1e6, "peak": peak, "unit": "GB/s",
                         "frac": bytes_it / ms_batch / 1e6 / peak, "traffic": None, "peak_source": peak_src,
                         "note": "algorithmic bytes of all iterations of all right-hand sides / whole-solve time; "
                                 "L2-resident for small grids, where the fraction is not an HBM statement"},
            "e2e": {"value": ms_e2e * 1e-3, "unit": UNIT, "h2d_bytes_per_step": int(B.nbytes), "d2h_bytes_per_step": int(B.nbytes)},
            "gpu_launches": 2 * args.steps, "clocks": clocks,
            "loop": ("one cluster-resident solve per right-hand side (k_pcg_cluster)" if cu.cuth_loop_home(g, opts) == 3
                     else "persistent cooperative kernel, lock-step over the right-hand sides (k_pcg_batch)")}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--grid", type=int, nargs=3, default=None, metavar=("NX", "NY", "NZ"),
                    help="the recipe of --config on another grid (for studying the automatic kernel choices)")
    ap.add_argument("--precision", default=None, choices=["fp64", "mixed"])
    ap.add_argument("--impl", default="cuth", choices=["cuth", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-window", action="store_true",
                    help="cpu_baseline from two timing windows instead of one full oracle solve (cfg 1, 2, 3, 6)")
    ap.add_argument("--no-cfg4", action="store_true",
                    help="default run (config 3) only: skip the appended block that solves BASELINE configs[3] "
                         "(4096x4096x8) once per precision")
    ap.add_argument("--kernel-reps", type=int, default=20)
    ap.add_argument("--preconditioner", default="jacobi", choices=["jacobi", "chebyshev"],
                    help="jacobi = the north_star hot path; chebyshev = the paper's own preconditioner (Alg. 3)")
    ap.add_argument("--cheb-degree", type=int, default=30)
    ap.add_argument("--lanczos-steps", type=int, default=40)
    ap.add_argument("--cheb-storage", default="fp32", choices=["fp32", "fp16"],
                    help="MIXED Chebyshev: matrix copy the preconditioner reads (A2 fp32 / A3 fp16, Alg. 4)")
    ap.add_argument("--transient-steps", type=int, default=0, help="config 5: time steps per bench step (default 200)")
    ap.add_argument("--cheb-fusion", type=int, default=0, choices=[0, 1, 2, 3],
                    help="cuth_tuning_t.cheb_fusion: 0 auto, 1 one Chebyshev pass per kernel, 2 two passes per kernel, 3 = 2 without TMA")
    ap.add_argument("--pair-occupancy", type=int, default=0, choices=[0, 2, 3, 4],
                    help="cuth_tuning_t.pair_occupancy: resident CTAs/SM of the TMA two-pass Chebyshev kernel (0 auto)")
    ap.add_argument("--pair-rows", type=int, default=0, choices=[0, 8, 16],
                    help="cuth_tuning_t.pair_rows: region height of the TMA two-pass Chebyshev kernel (0 auto)")
    ap.add_argument("--traversal", type=int, default=0, choices=[0, 1, 2],
                    help="cuth_tuning_t.traversal: 0 auto, 1 flat (3 kernels/iteration), 2 z-marching fused (2 kernels)")
    ap.add_argument("--profile-iters", type=int, default=0,
                    help="after the timed solves, replay this many loop bodies kernel by kernel OUTSIDE the "
                         "graph (ncu cannot see kernel nodes of graphs with conditional nodes)")
    ap.add_argument("--loop-mode", type=int, default=0, choices=[0, 1, 2, 3, 4],
                    help="cuth_tuning_t.loop_mode: 0 automatic, 1 CUDA graph, 2 persistent kernel wherever the flat traversal applies, "
                         "3 cluster-resident kernel, 4 its shared-memory form")
    ap.add_argument("--k1-variant", type=int, default=0, choices=[0, 1, 2, 3],
                    help="cuth_tuning_t.k1_variant: 0 auto, 1 one column per thread, 2 two columns (TMA-staged K1 when "
                         "nx %% 4 == 0), 3 two columns with ordinary loads")
    ap.add_argument("--lanczos-fp32", action="store_true",
                    help="Chebyshev setup: the paper's fp32 Lanczos on A2 (PAPER.md:340) instead of fp64 on A1")
    ap.add_argument("--batch", type=int, default=0,
                    help="NRHS > 0: time cuth_pcg_solve_batch on NRHS power maps of --config (FP64, Jacobi) against "
                         "NRHS single solves")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.batch > 0:
        import paper_2606_17850_b200 as cu0
        cu0.set_default_tuning(traversal=args.traversal, loop_mode=args.loop_mode, k1_variant=args.k1_variant)
        return run_batch(args)

    import torch
    import torch.distributed as dist
    import paper_2606_17850_b200 as cu

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the cuth path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # kernel variants travel in every call's cuth_tuning_t (the library has no process-wide settings)
    cu.set_default_tuning(traversal=args.traversal, loop_mode=args.loop_mode, cheb_fusion=args.cheb_fusion,
                          k1_variant=args.k1_variant, lanczos_fp32=1 if args.lanczos_fp32 else 0,
                          pair_occupancy=args.pair_occupancy, pair_rows=args.pair_rows)
    w = W.make_workload(args.config) if args.grid is None else \
        W.make_workload(args.config, nx=args.grid[0], ny=args.grid[1], nz=args.grid[2], n_hot=16)
    mixed = w.mixed if args.precision is None else (args.precision == "mixed")
    prec = cu.MIXED if mixed else cu.FP64
    kap = w.kappa_cell if w.kappa_cell is not None else w.kappa_layer
    kap_d = torch.from_numpy(np.ascontiguousarray(kap)).cuda()
    g = cu.Grid(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, kap_d, w.h_top, w.cvol, w.dt)
    A = cu.DiaMatrix(g)
    opts = cu.Opts(precision=prec, rtol=w.rtol, max_iters=200000, true_resid_period=w.true_resid_period)
    S = cu.Solver(A, opts)
    stream = torch.cuda.current_stream()

    # Inputs.  Steady: one power map b.  Transient (cfg 5): the whole trace of n_steps power maps, each
    # backward-Euler step warm-started from the previous one; ONE bench step = the whole trace.
    nt = 1
    if w.transient:
        nt = args.transient_steps or w.n_steps
        maps = [W.power_for_step(w, s + 1) for s in range(nt)]
        b_host = torch.from_numpy(np.stack(maps)).pin_memory()
        del maps
    else:
        b_host = torch.from_numpy(w.power).reshape(1, -1).pin_memory()
    x_host = torch.empty(w.n, dtype=torch.float64).pin_memory()
    b = b_host.cuda()
    b_stage = torch.empty(w.n, dtype=torch.float64, device="cuda")
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    cheb = args.preconditioner == "chebyshev"
    setup_ms = 0.0
    if cheb:       # setup: Lanczos on the device + tridiagonal eigenvalues on the host, once per matrix
        torch.cuda.synchronize()
        t0 = time.time()
        bounds = S.setup_chebyshev(b[0], lanczos_steps=args.lanczos_steps, degree=args.cheb_degree,
                                   storage=cu.CHEB_A3_FP16 if args.cheb_storage == "fp16" else cu.CHEB_DEFAULT)
        setup_ms = (time.time() - t0) * 1e3
    counters = torch.zeros(4, dtype=torch.int32, device="cuda")     # status, iterations, promotions, evals
    early_acc = torch.zeros(1, dtype=torch.int32, device="cuda")   # iterations done on the fp32-stored operator
    res_i32 = S.result_dev.view(torch.int32)

    def one_pass(from_host):
        """One bench step: x0 = 0, then the solve (steady) or the nt-step trace (transient)."""
        x.zero_()
        counters.zero_()
        early_acc.zero_()
        for s in range(nt):
            if from_host:
                b_stage.copy_(b_host[s], non_blocking=True)
                src = b_stage
            else:
                src = b[s]
            if w.transient:
                S.step(src, x)
            else:
                S.solve(src, x)
            counters.add_(res_i32[:4])
            if mixed:
                early_acc.add_(torch.where(res_i32[2:3] > 0, res_i32[9:10], res_i32[1:2]))
        if from_host:
            x_host.copy_(x, non_blocking=True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (value)
    for _ in range(args.warmup):
        one_pass(False)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for e0, e1 in ev:
        e0.record(stream)
        one_pass(False)
        e1.record(stream)
    barrier()
    clocks = sampler.stop() if sampler else None
    res = S.result()                       # record of the last solve / last time step
    cnt = counters.cpu().numpy()
    total_its, total_promos, total_evals, worst_status = int(cnt[1]), int(cnt[2]), int(cnt[3]), int(cnt[0])
    ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    ms_per_step = max_over_ranks(float(np.mean(ms)), world, "cuda")

    # ---- end-to-end through the public API with HOST buffers (pinned), copies inside the timed region
    barrier()
    e2e_ms = []
    for _ in range(max(1, min(args.steps, 3))):
        t0 = torch.cuda.Event(enable_timing=True)
        t1 = torch.cuda.Event(enable_timing=True)
        t0.record(stream)
        one_pass(True)
        t1.record(stream)
        torch.cuda.synchronize()
        e2e_ms.append(t0.elapsed_time(t1))
    e2e_ms_max = max_over_ranks(float(np.mean(e2e_ms)), world, "cuda")
    x_final = x_host.numpy().copy()

    # ---- dominant kernels timed one by one with CUDA events (same launch configuration as in the graph)
    peak, peak_src = peaks()
    lpi = cu.cuth_launches_per_iteration(g, S.opts)
    persistent = (lpi == 0) and not cheb                  # whole solve = one cooperative kernel
    fused = lpi > 0 and cu.cuth_traversal(g, S.opts) == 2     # z-marching graph loop: K1 (one or two nodes) + K2
    kern = {}

    def time_kernel(kid):
        for _ in range(3):
            cu.cuth_profile_kernel(S.work, g, S.opts, kid)
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.kernel_reps):
            cu.cuth_profile_kernel(S.work, g, S.opts, kid)
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.kernel_reps

    # The profile hook replays the loop-body kernels on the context the finished solve left in the workspace.  A MIXED
    # solve ends in the late stage (fp64 operator): -1 arms that; -2 re-arms the EARLY stage so that the fp32-stored
    # instantiation of K1 / the SpMV -- the one that ran most of the launches -- is timed as well.
    cu.cuth_profile_kernel(S.work, g, S.opts, -1)
    names = ({4: "k_fused_pspmv", 5: "k_update_nox", 3: "k_true_resid"} if fused else
             {0: "k_pupdate", 1: "k_spmv_dot", 2: "k_update", 3: "k_true_resid"})
    body_ids = (4, 5) if fused else (0, 1, 2)
    stage_tag = "fp64"
    if cheb:
        h16 = mixed and args.cheb_storage == "fp16"
        cid = 8 if h16 else (7 if mixed else 6)
        names[cid] = "k_cheb_mid"
        cheb_launches, cheb_npairs = cu.cuth_cheb_launches(g, S.opts)
        pid = 10 if h16 else 9                            # two passes per launch (cuth_tuning_t.cheb_fusion)
        # replay of one apply for ncu's launch list: the two-pass launches, and a single pass standing in for
        # each of FIRST / leftover MID / LAST (same stencil, same traffic to within 8 B/row)
        body_ids = tuple([pid] * cheb_npairs + [cid] * (cheb_launches - cheb_npairs)) + body_ids
        if mixed and w.nx % 2 == 0:
            names[pid] = "k_cheb_pair"
    a_kid = 4 if fused else 1                             # the kernel that applies A in the loop body
    a_name = names[a_kid]
    for kid, nm in names.items():
        kern[nm + ("[fp64 operator]" if kid == a_kid else "")] = time_kernel(kid)
    for _ in range(args.profile_iters):
        for kid in body_ids:
            cu.cuth_profile_kernel(S.work, g, S.opts, kid)
    if mixed and not cheb:
        cu.cuth_profile_kernel(S.work, g, S.opts, -2)
        kern[a_name + "[fp32-stored operator]"] = time_kernel(a_kid)
        if fused:
            kern["k_update_nox[early stage: fp32 1/D0, 28 B/row]"] = time_kernel(5)
        for _ in range(args.profile_iters):
            for kid in body_ids:
                cu.cuth_profile_kernel(S.work, g, S.opts, kid)
    torch.cuda.synchronize()
    # standalone SpMV (cuth_spmv), both precisions
    y = torch.empty_like(x)
    spmv = {}
    for nm, pr in (("fp64", cu.FP64), ("mixed", cu.MIXED)):
        for _ in range(3):
            cu.cuth_spmv_tuned(A.buf, g, pr, None, b[0], y)
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.kernel_reps):
            cu.cuth_spmv_tuned(A.buf, g, pr, None, b[0], y)
        e1.record(stream)
        torch.cuda.synchronize()
        tms = e0.elapsed_time(e1) / args.kernel_reps
        gbs = bytes_per_row(w, "spmv_" + nm) * w.n / tms / 1e6
        spmv[nm] = {"ms": tms, "gbs": gbs, "frac": gbs / peak, "frac_of_8TBs_nominal": gbs / 8000.0}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    it = total_its
    early = int(early_acc.item()) if mixed else 0
    late = it - early
    iter_bytes = (early * bytes_per_row(w, "iter_mixed_fused" if fused else "iter_mixed")
                  + late * bytes_per_row(w, "iter_fp64_fused" if fused else "iter_fp64")) * w.n
    m = m_ratio(w)
    if cheb:
        # outer: K1 (matrix + z, p, x read + p', mu, x written) + K2 (r, mu read, r written); preconditioner:
        # FIRST M+8+3s (2s in fp64), (k-3) x MID M+4s, LAST M+2s+16 with s = sizeof(T), M = matrix bytes per row
        #
        # a two-pass launch (k_cheb_pair_f32) moves M + 5s for two MID passes
        k, sT = args.cheb_degree, (4 if mixed else 8)
        Mc = (2 * (m - 1) if h16 else 4 * (m - 1)) if mixed else 8 * m
        singles = (k - 3) - 2 * cheb_npairs
        first_b, last_b = Mc + (3 if mixed else 2) * sT + 8, Mc + 2 * sT + 16
        if singles < 0:     # the odd MID pass shares its launch with LAST: U, V, r32, r read, z written (M + 3s + 16)
            apply_bytes = first_b + (cheb_npairs - 1) * (Mc + 5 * sT) + (Mc + 3 * sT + 16)
        else:
            apply_bytes = first_b + singles * (Mc + 4 * sT) + cheb_npairs * (Mc + 5 * sT) + last_b
        outer = lambda M_: M_ + 48 + 24          # no 1/D0 anywhere: z = q(A) r is a stored vector
        iter_bytes = (early * (outer(4 * (m - 1)) + apply_bytes) + late * (outer(8 * m) + apply_bytes)) * w.n
    iter_gbs = iter_bytes / (ms_per_step * 1e-3) / 1e9
    # The roofline line describes the instantiation that ran the MAJORITY of the launches of the timed solve.
    early_major = mixed and not cheb and early > late
    stage_tag = "fp32-stored" if early_major else "fp64"
    if fused:      # K1: matrix + r, p, x read + p', mu, x written (+ 1/D0 read with the fp32-stored operator)
        dom_name = "k_fused_pspmv"
        dom_bytes = ((4 * (m - 1) + 52) if early_major else (8 * m + 48)) * w.n
    else:
        dom_name = "k_spmv_dot"
        dom_bytes = bytes_per_row(w, "spmv_mixed" if early_major else "spmv_fp64") * w.n
    dom_ms = kern["%s[%s operator]" % (dom_name, stage_tag)]
    if cheb:
        dom_name, dom_ms = "k_cheb_mid", kern["k_cheb_mid"]
        dom_bytes = (((2 if h16 else 4) * (m - 1) + 16) if mixed else (8 * m + 32)) * w.n
        if cheb_npairs > 0:
            dom_name, dom_ms = "k_cheb_pair", kern["k_cheb_pair"]
            dom_bytes = ((2 if h16 else 4) * (m - 1) + 20) * w.n
        stage_tag = "fp32-stored" if mixed else "fp64"
    per_it = (lpi if fused else 3) + (cheb_launches if cheb else 0)
    per_eval = 3 if fused else 2
    launches = args.steps * (nt * (1 + 1 + 1 + (1 if w.transient else 0)) + per_it * it + per_eval * total_evals)
    if persistent:
        launches = args.steps * nt * (2 + (1 if w.transient else 0))      # k_set_ctx + k_pcg_persistent

    line = {
        "metric": METRIC, "value": ms_per_step * 1e-3, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "n_unknowns": w.n, "grid": [w.nx, w.ny, w.nz],
                   "precision": "mixed" if mixed else "fp64", "rtol": w.rtol, "preconditioner": args.preconditioner,
                   **({"cheb_degree": args.cheb_degree, "lanczos_steps": args.lanczos_steps,
                       "cheb_interval": [S.opts.cheb_lmin, S.opts.cheb_lmax], "cheb_storage": args.cheb_storage} if cheb else {}),
                   "l2_policy": ("inputs larger than L2 (matrix + vectors = %.2f GB streamed per iteration)" if
                                 (8 * m_ratio(w) + 48) * w.n > 126e6 else
                                 "working set %.3f GB fits the 126 MB L2: L2-resident, latency-bound case, "
                                 "no flush; HBM fractions are not meaningful here") %
                                ((8 * m_ratio(w) + 48) * w.n / 1e9),
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "iterations": it, "iterations_early_stage": early, "promotions": total_promos, "true_resid_evals": total_evals,
        "time_steps": nt,
        "switch_reason": res.switch_reason, "switch_mask": res.switch_mask, "switch_iteration": res.switch_iteration,
        "hard_restarts": res.hard_restarts, "soft_restarts": res.soft_restarts,
        "rel_resid_true": res.rel_resid_true, "status": res.status_name if worst_status == 0 else "not all steps converged",
        "us_per_iteration": ms_per_step * 1e3 / max(it, 1),
        "solves_per_s": world / (ms_per_step * 1e-3),
        "roofline": {"bound": "hbm", "kernel": "%s (%s operator; ran %d of the %d iterations)" %
                                               (dom_name, stage_tag, early if early_major else late, it),
                     "achieved": dom_bytes / dom_ms / 1e6, "peak": peak, "unit": "GB/s",
                     "frac": dom_bytes / dom_ms / 1e6 / peak, "frac_of_8TBs_nominal": dom_bytes / dom_ms / 1e6 / 8000.0,
                     "traffic": NCU_TRAFFIC_BYTES.get((w.name, dom_name, "mixed" if stage_tag == "fp32-stored" else "fp64")),
                     "peak_source": peak_src,
                     "ms_per_launch": dom_ms, "algorithmic_bytes_per_launch": dom_bytes},
        "roofline_iteration": {"bound": "hbm", "achieved": iter_gbs, "peak": peak, "unit": "GB/s",
                               "frac": iter_gbs / peak, "frac_of_8TBs_nominal": iter_gbs / 8000.0,
                               "algorithmic_bytes_per_solve": iter_bytes,
                               "note": ("Chebyshev: outer K1+K2 plus (k-1)-kernel apply bytes per row per iteration " if cheb else "") +
                                       "floor bytes (8m+88 fp64 three-kernel, 8m+80 fp64 fused / 4(m-1)+80 fp32-stored fused, 4(m-1)+88 unfused, per row per iteration) "
                                       "x iterations / whole-solve time, true-residual checks included in the time"},
        "kernels_ms": kern, "spmv": spmv, "setup_ms": setup_ms,
        "loop": {1: "cuda graph (conditional WHILE/IF nodes, %d iterations per pass)" % ((next((u for u in (10, 8, 6, 5, 4, 3) if w.true_resid_period % u == 0), 4) if mixed else 8) if fused and not cheb else 1),
                 2: "persistent cooperative kernel", 3: "cluster-resident kernel (one thread-block cluster)",
                 4: "fixed-FP32 ablation kernel"}[cu.cuth_loop_home(g, S.opts)],
        "e2e": {"value": e2e_ms_max * 1e-3, "unit": UNIT, "h2d_bytes_per_step": int(w.n * 8 * nt),
                "d2h_bytes_per_step": int(w.n * 8)},
        "gpu_launches": int(launches), "clocks": clocks,
    }
    if fused and not cheb:      # the other K1 instantiation, for the record
        for tag, nb in (("fp64", 8 * m + 48), ("fp32-stored", 4 * (m - 1) + 52)):
            key = "k_fused_pspmv[%s operator]" % tag
            if key in kern:
                gbs = nb * w.n / kern[key] / 1e6
                line.setdefault("k1_instantiations", {})[tag] = {"ms": kern[key], "gbs": gbs, "frac": gbs / peak,
                                                                "frac_of_8TBs_nominal": gbs / 8000.0, "bytes_per_row": nb}
        gbs = 32 * w.n / kern["k_update_nox"] / 1e6
        line["k2"] = {"ms": kern["k_update_nox"], "gbs": gbs, "frac": gbs / peak, "bytes_per_row": 32}
    if not args.no_cpu_baseline and world == 1:
        keep = {}
        line["cpu_baseline"] = cpu_oracle_baseline(w, args.config, x_gpu=None if w.transient else x_final,
                                                   full=False if args.cpu_window else None, out=keep)
        if not w.transient:
            # property check of the timed result against the ORACLE's matrix (not timed)
            from oracle import oracle as O
            Ao, bb = keep["A"], keep["b"]
            line["oracle_true_rel_resid_of_gpu_x"] = float(np.linalg.norm(bb - O.spmv(Ao, x_final)) / np.linalg.norm(bb))
        del keep
    if args.config == 3 and world == 1 and not args.no_cfg4 and not cheb:
        # the 134 M-unknown scaling case of BASELINE.json, one timed solve per precision, in the same record
        del S, A, b, b_stage, x, y, kap_d
        torch.cuda.empty_cache()
        line["cfg4"] = cfg4_block(cu, args, peak)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def cfg4_block(cu, args, peak):
    """BASELINE.json configs[3] (4096x4096x8, 134 M unknowns): ONE timed solve in FP64 and one in MIXED (after a
    5-iteration solve that instantiates the graph), the loop-body kernels and cuth_spmv timed as in the main record,
    and the true residual of the GPU's x recomputed with the ORACLE's CSR matrix."""
    import torch
    w = W.make_workload(4)
    g = cu.Grid(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, torch.from_numpy(np.ascontiguousarray(w.kappa_layer)).cuda(), w.h_top)
    A = cu.DiaMatrix(g)
    b = torch.from_numpy(w.power).cuda()
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    m = m_ratio(w)
    out = {"workload": w.name, "n_unknowns": w.n, "grid": [w.nx, w.ny, w.nz], "rtol": w.rtol}
    xs = {}
    for name, prec in (("fp64", cu.FP64), ("mixed", cu.MIXED)):
        S = cu.Solver(A, cu.Opts(precision=prec, rtol=w.rtol, max_iters=5, true_resid_period=w.true_resid_period))
        S.solve(b, x.zero_())                      # warm-up: graph instantiation, 5 iterations
        S.opts.max_iters = 200000
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        x.zero_()
        e0.record(stream)
        S.solve(b, x)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        r = S.result()
        early = (r.switch_iteration if r.promotions else r.iterations) if prec == cu.MIXED else 0
        ib = (early * (4 * (m - 1) + 80) + (r.iterations - early) * (8 * m + 80)) * w.n
        d = {"value": ms * 1e-3, "unit": UNIT, "iterations": r.iterations, "iterations_early_stage": early,
             "status": r.status_name, "rel_resid_true": r.rel_resid_true, "true_resid_evals": r.true_resid_evals,
             "switch_reason": r.switch_reason, "us_per_iteration": ms * 1e3 / max(r.iterations, 1),
             "roofline_iteration": {"achieved": ib / ms / 1e6, "unit": "GB/s", "frac": ib / ms / 1e6 / peak,
                                    "frac_of_8TBs_nominal": ib / ms / 1e6 / 8000.0}}

        def tk(kid):
            for _ in range(2):
                cu.cuth_profile_kernel(S.work, g, S.opts, kid)
            t0 = torch.cuda.Event(enable_timing=True)
            t1 = torch.cuda.Event(enable_timing=True)
            t0.record(stream)
            for _ in range(10):
                cu.cuth_profile_kernel(S.work, g, S.opts, kid)
            t1.record(stream)
            torch.cuda.synchronize()
            return t0.elapsed_time(t1) / 10

        x_keep = x.clone()
        cu.cuth_profile_kernel(S.work, g, S.opts, -1)
        k1, k2 = tk(4), tk(5)
        d["k1_fp64"] = {"ms": k1, "gbs": (8 * m + 48) * w.n / k1 / 1e6, "frac": (8 * m + 48) * w.n / k1 / 1e6 / peak}
        d["k2"] = {"ms": k2, "gbs": 32 * w.n / k2 / 1e6, "frac": 32 * w.n / k2 / 1e6 / peak}
        if prec == cu.MIXED:
            cu.cuth_profile_kernel(S.work, g, S.opts, -2)
            k1e = tk(4)
            d["k1_fp32_stored"] = {"ms": k1e, "gbs": (4 * (m - 1) + 52) * w.n / k1e / 1e6,
                                   "frac": (4 * (m - 1) + 52) * w.n / k1e / 1e6 / peak}
        xs[name] = x_keep.cpu().numpy()
        del x_keep
        S.close()
        del S
        out[name] = d
    y = torch.empty_like(x)
    for nm, pr, bpr in (("fp64", cu.FP64, 8 * m + 16), ("mixed", cu.MIXED, 4 * (m - 1) + 16)):
        for _ in range(2):
            cu.cuth_spmv_tuned(A.buf, g, pr, None, b, y)
        t0 = torch.cuda.Event(enable_timing=True)
        t1 = torch.cuda.Event(enable_timing=True)
        t0.record(stream)
        for _ in range(10):
            cu.cuth_spmv_tuned(A.buf, g, pr, None, b, y)
        t1.record(stream)
        torch.cuda.synchronize()
        tms = t0.elapsed_time(t1) / 10
        out.setdefault("spmv", {})[nm] = {"ms": tms, "gbs": bpr * w.n / tms / 1e6, "frac": bpr * w.n / tms / 1e6 / peak,
                                          "frac_of_8TBs_nominal": bpr * w.n / tms / 1e6 / 8000.0}
    del A, b, x, y
    torch.cuda.empty_cache()
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        Ao = O.assemble_workload(w)
        bn = np.linalg.norm(w.power)
        for name in ("fp64", "mixed"):
            out[name]["oracle_true_rel_resid_of_gpu_x"] = float(np.linalg.norm(w.power - O.spmv(Ao, xs[name])) / bn)
        out["max_abs_diff_mixed_vs_fp64_K"] = float(np.abs(xs["mixed"] - xs["fp64"]).max())
    return out


if __name__ == "__main__":
    main()
