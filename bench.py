#!/usr/bin/env python
"""bench.py -- pair-updates/s of the convex-clustering MM hot path (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

Workload (default `large_sparse` = BASELINE.json configs[3], the largest sparse single-GPU config and
the one north_star's roofline target names): seeded synthetic data from paper_1409_2065_b200.synth;
the k-NN Gaussian graph is built on the GPU by cc_knn_weights (a0).

One STEP = one cc_solve of `--iters` MM iterations (rows a1-a6 of DESIGN.md: right-hand side, CG
projection, pair norms + d_m + Phi, U update + shrink) at the next gamma of the 50-value grid, walked
with stride 5 and warm-started from the previous step, exactly as cc_path does.  One pair-update = one
undirected pair carried through one full MM iteration, projection sweeps included.

value   : |E| * iters * K / device time of the K steps, inputs resident in HBM.
e2e     : the same work through the C ABI starting from pinned HOST buffers: per step H2D of X and the
          CSR graph, cc_create, cc_solve, cc_get_U into host memory, cc_destroy.
roofline: the SWEEP (a1 right-hand side, a2 one inner projection sweep = k_cg_spmv +
          k_cg_update, a3 pair norms, a5+a6 update) with the largest share of device time; durations are
          measured live inside the timed region by the library's device-side %globaltimer marks (the
          kernels are nodes of a CUDA graph with device-side WHILE loops, so host events cannot bracket
          them); bytes per launch are SURVEY 8(d)'s no-reuse formulas (`bytes_per_launch`), the
          implementation's own stream count is printed beside them (`impl_bytes`), and `per_iteration`
          is the whole MM iteration against the same peak.  `traffic` / `l2_bytes` are ncu's DRAM and L2
          bytes per launch of the dominant kernel from the capture named in profiles/r2_traffic.json.
cpu_baseline: the fp64 oracle (oracle/), as it stands, on the host cores, SURVEY 8(d)'s protocol on a
          bounded sample: the same generator at `--cpu-n` points, `--cpu-iters` MM iterations at the
          first, middle and last gamma with the CG back-end on all cores, then one iteration at the
          middle gamma on a single thread.  `--cpu-full` runs the protocol at the full size (minutes).
--impl reference: the oracle timed step by step on the same bounded sample (driver contract).
N > 1   : the path does not shard without a halo exchange: N independent
          replicas with different seeds, no collective on the data path, scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

GRID = {"large_sparse": (1.0, 1000.0, 50), "tiny": (1e-3, 1e3, 20), "expression": (0.05, 50.0, 40),
        "genotype": (1.0, 100.0, 50), "dense_weight": (1.0, 100.0, 30), "popres": (0.01, 10.0, 30)}
CPU_SAMPLE = {"large_sparse": lambda a: {"n": a.cpu_n}, "genotype": lambda a: {"p": 20000},
              "dense_weight": lambda a: {"n": 512}, "tiny": lambda a: {}, "expression": lambda a: {},
              "popres": lambda a: {}}
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # SMs x FP32 lanes x 2 flop/FMA x max clock (B200_PROFILING.md table)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="large_sparse", choices=list(GRID))
    ap.add_argument("--iters", type=int, default=20, help="MM iterations per step")
    ap.add_argument("--n", type=int, default=0, help="override the number of points (0 = config size)")
    ap.add_argument("--cpu-n", type=int, default=20000, help="points in the oracle's bounded sample (large_sparse)")
    ap.add_argument("--cpu-iters", type=int, default=3)
    ap.add_argument("--cpu-full", action="store_true", help="cpu_baseline at the full configuration size (minutes)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-path", action="store_true", help="skip the full gamma-path wall time")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--continuation-study", default="",
                    help="comma-separated stop tolerances (e.g. 1e-5,1e-6,1e-7): for each, the plain gamma path and the two staged "
                         "kappa schedules are timed and their U compared with a path converged at tol 1e-9 (adds minutes)")
    ap.add_argument("--eager", action="store_true", help="plain stream launches instead of the CUDA graph (for ncu)")
    return ap.parse_args()


def gamma_for_step(workload, step):
    from paper_1409_2065_b200 import synth
    lo, hi, ng = GRID[workload]
    grid = synth.gamma_grid(lo, hi, ng)
    return float(grid[(step * 5) % ng])


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thr.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in self.rows if len(r) >= 7 for k in range(4) if r[3 + k] == "Active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def cpu_count_used(O):
    return int(O.num_threads())


def _oracle_problem(args, full=False):
    """The workload's generator (bounded sample unless `full`), graph and weights by the oracle's own eq.-8 code."""
    from oracle import oracle as O
    from paper_1409_2065_b200 import synth
    O.build()
    wl = synth.make(args.workload, **({} if full else CPU_SAMPLE[args.workload](args)))
    X = wl.X.astype(np.float64)
    if wl.phi_rule == "fixed":
        phi = wl.phi
    else:
        si, sj = synth.sample_pairs(wl.n, 200_000, wl.seed)
        d2 = O.pair_dist2(X, wl.mask, si, sj)
        phi = 1.0 / float(np.median(d2[np.isfinite(d2)]))
    if wl.graph == "knn":
        ei, ej, w, _ = O.knn_graph(X, wl.mask, wl.k, phi)
    else:
        ei, ej, w, _ = O.complete_graph(X, wl.mask, phi)
    return O, wl, X, ei, ej, w


def oracle_sample(args, steps, warmup):
    """--impl reference: the oracle step by step on the bounded sample; returns (pair-updates/s, info, s per step)."""
    O, wl, X, ei, ej, w = _oracle_problem(args)
    U, V = O.cold_start(X, wl.mask, ei, ej)
    times = []
    for s in range(warmup + steps):
        g = gamma_for_step(args.workload, s)
        rho, eps = O.default_rho_eps(X, wl.mask, w, g)
        t0 = time.perf_counter()
        r = O.mm(X, wl.mask, ei, ej, w, g, rho, eps, U, V, args.cpu_iters, proj_method=1)
        dt = time.perf_counter() - t0
        U, V = r["U"], r["V"]
        if s >= warmup:
            times.append(dt)
    tot = float(sum(times))
    val = len(ei) * args.cpu_iters * len(times) / tot
    info = {"value": val, "unit": "pair-updates/s", "cores": cpu_count_used(O), "kind": "oracle",
            "sample": f"{args.workload} generator at n={wl.n}, p={wl.p} (|E|={len(ei)}), {len(times)} step(s) x "
                      f"{args.cpu_iters} MM iterations, fp64, explicit V, CG projection to 1e-13"}
    return val, info, tot / max(1, len(times))


def oracle_protocol(args, full=False):
    """cpu_baseline, SURVEY 8(d) "Timing the oracle beside it": `cpu_iters` MM iterations at the first, middle and last
    gamma of the grid (warm-started in that order, CG back-end) on all cores, then one iteration at the middle gamma on
    a single thread; core count read at run time.  Bounded sample of the workload unless `full`."""
    from paper_1409_2065_b200 import synth
    O, wl, X, ei, ej, w = _oracle_problem(args, full)
    lo, hi, ng = GRID[args.workload]
    grid = synth.gamma_grid(lo, hi, ng)
    gs = [float(grid[0]), float(grid[ng // 2]), float(grid[-1])]
    cores = cpu_count_used(O)
    U, V = O.cold_start(X, wl.mask, ei, ej)
    per_gamma, tot = [], 0.0
    mid_state = None
    for g in gs:
        rho, eps = O.default_rho_eps(X, wl.mask, w, g)
        if g == gs[1]:
            mid_state = (U, V, rho, eps)
        t0 = time.perf_counter()
        r = O.mm(X, wl.mask, ei, ej, w, g, rho, eps, U, V, args.cpu_iters, proj_method=1)
        dt = time.perf_counter() - t0
        U, V = r["U"], r["V"]
        tot += dt
        per_gamma.append({"gamma": g, "s_per_iteration": dt / args.cpu_iters, "cg_iterations_per_iteration": r["proj_cycles"] / args.cpu_iters})
    val = len(ei) * args.cpu_iters * len(gs) / tot
    O.set_threads(1)
    Um, Vm, rho, eps = mid_state
    t0 = time.perf_counter()
    O.mm(X, wl.mask, ei, ej, w, gs[1], rho, eps, Um, Vm, 1, proj_method=1)
    t1 = time.perf_counter() - t0
    O.set_threads(cores)
    return {"value": val, "unit": "pair-updates/s", "cores": cores, "kind": "oracle",
            "single_thread_value": len(ei) / t1, "per_gamma": per_gamma,
            "sample": f"{args.workload} generator at n={wl.n}, p={wl.p} (|E|={len(ei)}){' = the full configuration' if full else ''}: "
                      f"{args.cpu_iters} MM iterations at gamma = first/middle/last of the grid on {cores} threads, then 1 iteration "
                      f"at the middle gamma on 1 thread; fp64, explicit V, CG projection to 1e-13"}


def sweep_bytes(n, p, nnz, masked, dense=False):
    """SURVEY 8(d) algorithmic bytes per sweep, "no-reuse" model: every gathered neighbour row counts once per
    directed entry, own rows and outputs once per node; fp32.  Keys are the sweeps, values (bytes, kernels)."""
    npb, E = 4 * n * p, nnz // 2
    if dense and n <= 64:
        # genotype-like: read U, A', write A + read X, U, A, write U (SURVEY 8(d) "Dense path": 7 node arrays)
        # (the block soft-threshold over the n x n matrices, a4, rides in k_update's launch: 16 n^2 bytes)
        return {"a9_small": (7 * npb, ("kd_proj",)), "a5_update": (4 * npb + n * p + 16 * n * n, ("k_update",))}
    if dense:
        # dense-weight: W (n x n) once + ~10 node arrays per MM iteration; per kernel the n x n it must touch
        return {"a9_proj": (4 * n * n + 5 * npb, ("kd_proj",)), "a9_pairs": (4 * n * n // 2 + 2 * npb, ("kd_pairs",)),
                "a4_edges": (8 * n * n, ("kd_edges",)), "a5_update": (4 * npb + n * p, ("k_update",))}
    return {"a1_rhs": (nnz * (4 * p + 12) + 3 * npb, ("k_rhs",)),
            "a2_sweep": (nnz * (4 * p + 4) + 7 * npb, ("k_cg_spmv", "k_cg_update")),
            "a3_norms": (E * (8 * p + 12) + 2 * npb, ("k_norm",)),
            "a5_update": (4 * npb + n * p, ("k_update",))}


def impl_bytes(kernel, n, p, nnz, masked, dense=False):
    """What the kernels as written stream per launch (own count, for comparison with sweep_bytes)."""
    row, npb = 4 * p, 4 * n * p
    return {
        "k_rhs": nnz * (row + 8) + 5 * npb + 4 * n,          # z_j for every entry; a'_j only for unfused pairs (not counted)
        "k_cg_spmv": nnz * (row + 4) + 5 * npb + 4 * n,      # gather + own uc, p, s in; p, s out
        "k_cg_update": 6 * npb + 4 * n,                      # p, s, A, uc in; A, uc out
        "k_norm": (nnz // 2) * (2 * row + 28) + 4 * npb + (n * p if masked else 0) + 8 * n,
        # dense: A, U, X in, U and A' out -- n <= 64: no A' (the fused kernel reads A and dbar), + the n x n shrink
        "k_update": ((4 * npb + 16 * n * n if n <= 64 else 5 * npb) if dense else 8 * npb + 16 * nnz) + (n * p if masked else 0),
        # n <= 64: the fused kernel streams U, A', X in and A out.  Tensor-core path (n >= 128): kd_proj_tc3 reads the ratio
        # matrix R (n x n) + the pre-split B operand (2 np, re-read per row tile from L2) + 5 node arrays; kd_pairs_tc2 reads
        # ||b||, R, W of the upper triangle and writes ||b|| (upper) and R (both triangles) + the pre-split operands
        "kd_proj": (4 * npb if n <= 64 else 4 * n * n + 2 * npb + 5 * npb) + (n * p if masked else 0),
        "kd_pairs": 3 * npb + (n * n // 2) * 12 + (n * n // 2) * 4 + 4 * n * n,
        "kd_edges": 16 * n * n,
    }[kernel]


def alg_flops(kernel, n, p, dense_small):
    """Algorithmic floating-point operations per launch (FMA = 2): the contraction S.A' 2 n^2 p, the pair
    norms 6p per unordered pair; n <= 64: Gram-equivalent 2 n^2 p / 2 + contraction 2 n^2 p."""
    if dense_small:
        return {"kd_proj": 2.0 * n * n * p + 1.0 * n * n * p}.get(kernel, 0.0)
    return {"kd_proj": 2.0 * n * n * p, "kd_pairs": 2.0 * (n * (n - 1) / 2) * p}.get(kernel, 0.0)


def aggregate(dist, dev, times_ms, units):
    """Whole-job numbers from per-rank ones: MAX of the device times, SUM of the units processed.
    `dist` is torch.distributed (any backend) or None for a single process."""
    if dist is None:
        return [float(t) for t in times_ms], [float(u) for u in units]
    import torch
    t = torch.tensor(times_ms, device=dev, dtype=torch.float64)
    u = torch.tensor(units, device=dev, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return [float(x) for x in t], [float(x) for x in u]


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    val, info, s_per_step = oracle_sample(args, args.steps, args.warmup)
    line = {"impl": "reference", "metric": "pair-updates/sec per MM iteration", "value": val,
            "unit": "pair-updates/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * s_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": args.workload, "iters_per_step": args.cpu_iters},
            "cpu_baseline": info, "gpu_launches": 0,
            "e2e": {"value": val, "unit": "pair-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1409_2065_b200 import synth
    from paper_1409_2065_b200 import binding as B   # fails loudly when the CUDA library is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    kw = {"n": args.n} if args.n else {}
    wl = synth.make(args.workload, seed=rank, **kw)      # replicas differ by seed
    n, p = wl.n, wl.p
    Xh = torch.from_numpy(wl.X).pin_memory()
    Mh = None if wl.mask is None else torch.from_numpy(wl.mask).pin_memory()
    X = Xh.to(dev)
    M = None if Mh is None else Mh.to(dev)
    # phi rule S10: 1 / median squared distance over seeded sample pairs (torch only moves the data; the
    # median of ~2e5 numbers is input preparation, not a step of the path)
    if wl.phi_rule == "fixed":
        phi = wl.phi
    else:
        si, sj = synth.sample_pairs(n, 200_000, wl.seed)
        d = X[torch.from_numpy(si).to(dev)] - X[torch.from_numpy(sj).to(dev)]
        phi = 1.0 / float((d * d).sum(1).median())
    dense = wl.graph == "complete"
    t0 = time.perf_counter()
    if dense:
        Wd = B.cc_dense_weights(n, p, X, M, phi)
        rowptr = col = None
        w = Wd
        nnz = n * (n - 1)
    else:
        rowptr, col, w = B.cc_knn_weights(n, p, X, M, wl.k, phi)
        nnz = int(col.numel())
    torch.cuda.synchronize()
    t_knn = time.perf_counter() - t0
    if not dense:
        rowptr_h, col_h, w_h = rowptr.cpu().pin_memory(), col.cpu().pin_memory(), w.cpu().pin_memory()
    E = nnz // 2
    prm = B.cc_default_params(use_graph=0 if args.eager else 1, dense=1 if dense else 0)
    h = B.cc_create(n, p, X, M, rowptr, col, w, prm)
    for s in range(args.warmup):
        B.cc_solve(h, gamma_for_step(args.workload, s), 0.0, args.iters)
    small_sparse = (not dense) and n <= 384       # persistent single-kernel solve: its phase timing is a separate, untimed pass
    if not small_sparse:
        B.cc_reset_profile(h)
    launches0 = B.cc_get_counts(h)["launches"]
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev0.record()
    iters_done = 0
    for s in range(args.steps):
        it, _, _ = B.cc_solve(h, gamma_for_step(args.workload, args.warmup + s), 0.0, args.iters)
        iters_done += it
    ev1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop()
    stats = B.cc_get_stats(h)
    launches = B.cc_get_counts(h)["launches"] - launches0
    if small_sparse:          # the same steps again with the phase timers on (not inside the timed region: the timers cost time)
        B.cc_reset_profile(h)
        for s in range(args.steps):
            B.cc_solve(h, gamma_for_step(args.workload, args.warmup + s), 0.0, args.iters)
    prof = B.cc_get_profile(h)
    cg_per_it = prof["k_cg_spmv"]["calls"] / max(1, iters_done)
    prof = {k: v for k, v in prof.items() if v["calls"]}

    # ---- full gamma path (rank 0, N = 1): the other half of BASELINE.json's metric
    path = None
    if not args.no_path and world == 1:
        lo, hi, ng = GRID[args.workload]
        gam = [float(g) for g in synth.gamma_grid(lo, hi, ng)]
        B.cc_reset(h)
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record()
        its, _ = B.cc_path(h, gam, 1e-5, 2000)
        p1.record()
        torch.cuda.synchronize()
        lab = torch.empty(n, dtype=torch.int32, device=dev)
        ks = [B.cc_clusters(h, g, lab)[1] for g in (0, ng // 2, ng - 1)]
        path = {"n_gamma": ng, "gamma_lo": lo, "gamma_hi": hi, "tol": 1e-5, "maxit": 2000,
                "wall_s": p0.elapsed_time(p1) / 1e3, "iters_total": int(sum(its)),
                "nclusters_first_mid_last": ks}
        # the same path with kappa continuation (S26): same stop rule, same last stage
        Up = [torch.empty(n, wl.p, device=dev) for _ in range(3)]
        for u, g in zip(Up, (0, ng // 2, ng - 1)):
            B.cc_get_U(h, g, u)
        B.cc_reset(h)
        p0.record()
        its_c, _ = B.cc_path_continuation(h, gam, 0.1, 0.1, 200, 1e-5, 2000)
        p1.record()
        torch.cuda.synchronize()
        ks_c = [B.cc_clusters(h, g, lab)[1] for g in (0, ng // 2, ng - 1)]
        Uc = torch.empty(n, wl.p, device=dev)
        dU = []
        for u, g in zip(Up, (0, ng // 2, ng - 1)):
            B.cc_get_U(h, g, Uc)
            dU.append(float((Uc - u).norm() / u.norm().clamp_min(1e-30)))
        path["continuation"] = {"kappa_start": 0.1, "factor": 0.1, "stage_maxit": 200,
                                "wall_s": p0.elapsed_time(p1) / 1e3, "iters_total": int(sum(its_c)),
                                "nclusters_first_mid_last": ks_c, "rel_dU_vs_plain_first_mid_last": dU}
        del Up, Uc
        if args.continuation_study:
            # distance to the converged path (S26 / section 6 table): the reference is the plain iteration at tol 1e-9
            idx = sorted({ng // 4, ng // 2, (3 * ng) // 4, ng - 1})
            B.cc_reset(h)
            p0.record()
            its_r, _ = B.cc_path(h, gam, 1e-9, 20000)
            p1.record()
            torch.cuda.synchronize()
            ref_s = p0.elapsed_time(p1) / 1e3
            Ur = [B.cc_get_U(h, g, torch.empty(n, wl.p, device=dev)) for g in idx]
            Ut = torch.empty(n, wl.p, device=dev)

            def errs():
                out = []
                for u, g in zip(Ur, idx):
                    B.cc_get_U(h, g, Ut)
                    out.append(float((Ut - u).norm() / u.norm().clamp_min(1e-30)))
                return out
            rows = []
            for tol_s in args.continuation_study.split(","):
                tol = float(tol_s)
                row = {"tol": tol}
                for name, run in (("plain", lambda: B.cc_path(h, gam, tol, 20000)),
                                  ("staged_0.1_0.01", lambda: B.cc_path_continuation(h, gam, 0.1, 0.1, 200, tol, 20000)),
                                  ("staged_1_0.1_0.01", lambda: B.cc_path_continuation(h, gam, 1.0, 0.1, 200, tol, 20000))):
                    B.cc_reset(h)
                    p0.record()
                    its_x, _ = run()
                    p1.record()
                    torch.cuda.synchronize()
                    row[name] = {"wall_s": p0.elapsed_time(p1) / 1e3, "iters_total": int(sum(its_x)), "rel_err_vs_converged": errs()}
                rows.append(row)
            path["continuation_study"] = {"gamma_indices": idx, "reference": {"tol": 1e-9, "maxit": 20000, "wall_s": ref_s,
                                                                              "iters_total": int(sum(its_r))}, "rows": rows}
            del Ur, Ut
    B.cc_destroy(h)

    # ---- e2e: host buffers -> cc_create -> cc_solve -> U back on the host, every step
    e2e = None
    if not args.no_e2e:
        Uh = torch.empty(n, p, dtype=torch.float32).pin_memory()
        h2d = Xh.numel() * 4 + (Mh.numel() if Mh is not None else 0)
        if not dense:
            h2d += rowptr_h.numel() * 8 + col_h.numel() * 4 + w_h.numel() * 4
        d2h = Uh.numel() * 4

        def e2e_step(s):
            Xd = Xh.to(dev, non_blocking=True)
            Md = None if Mh is None else Mh.to(dev, non_blocking=True)
            if dense:   # the weights are rebuilt on the device from X: part of the user's call sequence
                rp = cl = None
                ww = B.cc_dense_weights(n, p, Xd, Md, phi)
            else:
                rp, cl, ww = rowptr_h.to(dev, non_blocking=True), col_h.to(dev, non_blocking=True), w_h.to(dev, non_blocking=True)
            hh = B.cc_create(n, p, Xd, Md, rp, cl, ww, B.cc_default_params(dense=1 if dense else 0))
            it, _, _ = B.cc_solve(hh, gamma_for_step(args.workload, s), 0.0, args.iters)
            B.cc_get_U(hh, -1, Uh)
            B.cc_destroy(hh)
            return it
        for s in range(2):
            e2e_step(s)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        it_e = sum(e2e_step(args.warmup + s) for s in range(args.steps))
        e1.record()
        torch.cuda.synchronize()
        ms_e = e0.elapsed_time(e1)
        e2e = {"ms": ms_e, "iters": it_e, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)}

    # ---- max over ranks, whole-job aggregate
    units = float(E) * iters_done
    units_e = float(E) * e2e["iters"] if e2e else 0.0
    (ms, ms_e2e), (units, units_e2e) = aggregate(dist if world > 1 else None, dev,
                                                 [ms, e2e["ms"] if e2e else 0.0], [units, units_e])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    peaks = json.load(open(peaks_path)) if os.path.exists(peaks_path) else {}
    if "hbm_gbs" in peaks:
        peak, peak_src = float(peaks["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    else:
        peak, peak_src = 6650.0, "B200_PROFILING.md fallback (of fallback)"
    # TF32 tensor peak = measured bf16 cuBLAS peak x the nominal tf32/bf16 ratio (1.1 / 2.25), B200_PROFILING.md; the
    # sustained figure, because the kernel is timed inside a long step
    bf16 = float(peaks.get("bf16_tflops_sustained", peaks.get("bf16_tflops", 1400.0)))
    tf32_peak = bf16 * 1.1 / 2.25
    masked = M is not None
    dense_small = dense and n <= 64
    # small n: the whole solve is one persistent kernel (cc_persist.cu); its timer slots are the phases of an iteration
    persistent = (not dense) and "k_cg_spmv" not in prof and "kd_proj" in prof
    if persistent:
        names = {"k_rhs": "phase1a_rhs", "k_cg_update": "phase1b_projection_by_inverse", "k_norm": "phase1c_norms_partials",
                 "k_update": "phase2_shrink_update", "kd_proj": "barrier_A_wait+scalars", "kd_pairs": "barrier_B_wait"}
        phases = {names[k]: {"us_per_iteration": v["ns"] / v["calls"] / 1e3} for k, v in prof.items() if k in names}
        prof = {}
    tot_ns = sum(v["ns"] for v in prof.values()) or 1.0
    per_kernel = {}
    for k, v in prof.items():
        dur = v["ns"] / v["calls"]
        per_kernel[k] = {"share": v["ns"] / tot_ns, "us_per_launch": dur / 1e3, "launches": v["calls"],
                         "impl_bytes": impl_bytes(k, n, p, nnz, masked, dense),
                         "impl_gbs": impl_bytes(k, n, p, nnz, masked, dense) / dur}
        fl = alg_flops(k, n, p, dense_small)
        if fl:
            per_kernel[k].update(alg_flops=fl, alg_tflops=fl / dur / 1e3)
    # sweeps of SURVEY 8(d): bytes by its formulas, time = the sweep's kernels together, per launch of the first one
    sweeps = {}
    for name, (nbytes, kernels) in sweep_bytes(n, p, nnz, masked, dense).items():
        if not all(k in prof for k in kernels):
            continue
        calls = prof[kernels[0]]["calls"]
        ns = sum(prof[k]["ns"] for k in kernels)
        sweeps[name] = {"kernels": list(kernels), "bytes_per_launch": nbytes, "us_per_launch": ns / calls / 1e3,
                        "launches": calls, "share": ns / tot_ns, "alg_gbs": nbytes / (ns / calls), "frac": nbytes / (ns / calls) / peak}
    it_us = 1e3 * ms / max(1, iters_done)
    if persistent:
        # SURVEY 8(d) bytes of one MM iteration with the projection by the precomputed inverse (Minv n x n + uc in, A out)
        sb = sweep_bytes(n, p, nnz, masked, dense)
        it_bytes = sb["a1_rhs"][0] + sb["a3_norms"][0] + sb["a5_update"][0] + 4 * n * n + 3 * 4 * n * p
        sweeps["mm_iteration"] = {"kernels": ["k_mm_persist"], "bytes_per_launch": it_bytes, "us_per_launch": it_us,
                                  "launches": iters_done, "share": 1.0, "alg_gbs": it_bytes / (it_us * 1e3),
                                  "frac": it_bytes / (it_us * 1e3) / peak}
    top = max(sweeps, key=lambda k: sweeps[k]["share"])
    topk = sweeps[top]["kernels"][0]
    it_bytes = sum(v["bytes_per_launch"] * v["launches"] for v in sweeps.values()) / max(1, iters_done)
    per_iteration = {"bytes": it_bytes, "us": it_us, "alg_gbs": it_bytes / (it_us * 1e3), "frac": it_bytes / (it_us * 1e3) / peak,
                     "note": "sum over the sweeps of SURVEY 8(d) bytes x launches / MM iterations, over the event-timed step"}
    # DRAM and L2 bytes per launch of the dominant kernel: from the committed ncu capture (provenance in the file)
    traffic = l2_bytes = tsrc = None
    tpath = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        ent = tj.get(args.workload, {}).get(topk)
        if ent:
            traffic, l2_bytes = ent.get("dram_bytes"), ent.get("lts_bytes")
            tsrc = {"capture": ent.get("capture"), "date": ent.get("date"), "command": tj.get("_command")}
    if dense and not dense_small and "kd_proj" in per_kernel:
        # dense-weight: the bound is the tensor pipe; useful flops = 2 n^2 p (contraction) + n^2 p (pair Grams,
        # symmetric) = 6p per unordered pair; 3xTF32 issues three MMAs per useful product (10 per K step in the pair kernel)
        tens = {k: per_kernel[k] for k in ("kd_proj", "kd_pairs") if k in per_kernel}
        fl_it = sum(v["alg_flops"] * v["launches"] for v in tens.values()) / max(1, iters_done)
        for k, v in tens.items():
            v["frac_tensor_useful"] = v["alg_tflops"] / tf32_peak
        tk = max(tens, key=lambda k: tens[k]["share"])
        roofline = {"bound": "tensor", "kernel": tk, "achieved": tens[tk]["alg_tflops"], "peak": tf32_peak, "unit": "TFLOP/s",
                    "frac": tens[tk]["alg_tflops"] / tf32_peak, "traffic": traffic, "l2_bytes": l2_bytes, "traffic_source": tsrc,
                    "peak_source": "TF32 = MEASURED_PEAKS.json bf16_tflops_sustained x 1.1/2.25 (nominal ratio; of measured)",
                    "flops_per_launch": tens[tk]["alg_flops"],
                    "per_iteration": {"flops": fl_it, "us": it_us, "alg_tflops": fl_it / it_us / 1e6, "frac": fl_it / it_us / 1e6 / tf32_peak,
                                      "hbm": per_iteration},
                    "note": "useful (algorithmic) flops; the 3xTF32 split issues 3 MMAs per product, so the tensor pipe is about 3x busier than frac says"}
    elif dense_small:
        # genotype-like: near the ridge: report against HBM (7 node arrays per iteration) and print the FP32 figure beside it
        v = per_kernel["kd_proj"]
        roofline = {"bound": "hbm", "kernel": "kd_small_tc", "achieved": sweeps[top]["alg_gbs"], "peak": peak, "unit": "GB/s",
                    "frac": sweeps[top]["frac"], "traffic": traffic, "l2_bytes": l2_bytes, "traffic_source": tsrc, "peak_source": peak_src,
                    "bytes_per_launch": sweeps[top]["bytes_per_launch"], "alg_tflops": v.get("alg_tflops"),
                    "frac_fp32_alu": v.get("alg_tflops", 0.0) / FP32_PEAK_TFLOPS, "per_iteration": per_iteration}
    else:
        roofline = {"bound": "hbm", "kernel": "+".join(sweeps[top]["kernels"]), "sweep": top, "achieved": sweeps[top]["alg_gbs"],
                    "peak": peak, "unit": "GB/s", "frac": sweeps[top]["frac"], "traffic": traffic, "l2_bytes": l2_bytes,
                    "traffic_source": tsrc, "peak_source": peak_src, "bytes_per_launch": sweeps[top]["bytes_per_launch"],
                    "per_iteration": per_iteration,
                    "note": ("latency-bound configuration (SURVEY 8(d): roofline % is not meaningful here): the state lives in shared "
                             "memory for the whole solve, one MM iteration = two grid barriers; the figure to read is us per iteration")
                            if persistent else
                            ("bytes are SURVEY 8(d)'s no-reuse algorithmic figures; the gathered arrays are L2-resident, so a fraction "
                             "near or above 1 of the HBM copy peak reads as an L2-served gather (see traffic vs l2_bytes), not as HBM "
                             "bandwidth")}
    roofline.update(timing="device %globaltimer marks inside the timed region (kernel + launch gap)", sweeps=sweeps,
                    kernels=phases if persistent else per_kernel, device_ms_sum=tot_ns / 1e6)

    line = {"metric": "pair-updates/sec per MM iteration", "value": units / (ms / 1e3), "unit": "pair-updates/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload,
                       "workload_note": "large_sparse is the config north_star names for the roofline target and the largest sparse "
                                        "single-GPU one; other configs: --workload (numbers in profiles/)",
                       "n": n, "p": p, "k": wl.k, "pairs": E, "nnz": nnz,
                       "iters_per_step": args.iters, "gamma": "50-value log grid walked with stride 5, warm-started",
                       "cg_sweeps_per_iter": cg_per_it, "rho": stats["rho"], "kappa": 1e-2, "proj_tol": 1e-5,
                       "l2": "working set (node arrays + pair arrays, %.0f MB) vs 126 MB L2; no flush" %
                             ((10 * n * p * 4 + (16 * n * n if dense else 24 * nnz)) / 1e6),
                       "parallelism": "replicas" if world > 1 else "single", "knn_build_s": t_knn},
            "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline}
    if e2e:
        line["e2e"] = {"value": units_e2e / (ms_e2e / 1e3), "unit": "pair-updates/s",
                       "h2d_bytes_per_step": e2e["h2d_bytes_per_step"], "d2h_bytes_per_step": e2e["d2h_bytes_per_step"],
                       "ms_per_step": ms_e2e / args.steps}
    if path:
        line["path"] = path
    if not args.no_cpu and world == 1:
        try:
            line["cpu_baseline"] = oracle_protocol(args, full=args.cpu_full)
        except Exception as ex:  # the baseline is reported, never required for the GPU number
            line["cpu_baseline"] = {"value": None, "unit": "pair-updates/s", "cores": os.cpu_count(), "kind": "oracle",
                                    "sample": f"failed: {ex}"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
