#!/usr/bin/env python
"""bench.py -- BSE block-apply throughput on one B200 (BASELINE.json metric), with roofline, e2e and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--k 4] [--impl reference]

A "step" is one bse_apply (Y = R X, k columns) over the packed triangular operator of the chosen BASELINE.json
config (default: config 4, TDA N = 98304, 77 GB -- the largest single-GPU configuration; the operand is ~600x
larger than L2, so no flush is needed between iterations).  `value` is algorithmic GB/s: (packed matrix bytes +
32 N k) / time, whole job.  Extra keys report the k sweep, the Lanczos time-to-nev at config 2, the roofline of the
apply kernel, the end-to-end number through the host entry point, and the CPU oracle timed on the host cores.
Multi-GPU (torchrun): the path does not shard (north_star: one GPU) -- N independent replicas, scaling "weak".
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

import bse_inputs as gen  # noqa: E402

METRIC = "bse_block_apply_algorithmic_GBps"
UNIT = "GB/s"


ES = 16.0      # bytes per stored entry; --storage c64 sets 8 (complex64-stored operand)


def alg_bytes(N: int, k: int) -> float:
    """B_mat + 32 N k  (packed lower triangle once, X read + Y written; complex128 vectors)."""
    return ES * N * (N + 1) / 2 + 32.0 * N * k


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def max_over_ranks(value: float, dist, device) -> float:
    """Timing of a multi-rank run is the MAX over ranks (every rank is an independent replica)."""
    if dist is None:
        return value
    import torch
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def time_steps(fn, steps, warmup):
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps      # ms per step, on the stream the kernels were launched on


def cpu_oracle_sample(N, k, group, seed, sample_rows, reps):
    """The oracle as it stands, timed on the host cores on a bounded sample: `sample_rows` full rows of R (from the CPU
    generator) times the X block.  Returns (seconds per repetition, threads).  Only this leg and --impl reference
    may touch oracle/."""
    import oracle
    oracle.build()
    rows = (np.arange(sample_rows, dtype=np.int64) * 2654435761 % N)
    Hrows = gen.rows_R(N, seed, rows, 0.0, group)
    if ES == 8.0:
        Hrows = oracle.round_c64(Hrows)            # the complex64-stored operator is the rounded matrix
    X = gen.block_X(N, k, seed + 1000)
    oracle.rows_times_block(Hrows[:8], X)          # warm the library
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle.rows_times_block(Hrows, X)
    return (time.perf_counter() - t0) / reps, oracle.num_threads()


def run_reference(args, cfg):
    """--impl reference: for this tier the reference arm is the CPU oracle (no installable reference exists: the
    reference is a paper).  One step = the oracle's dense row-panel product on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    N, k = cfg["N"], args.k
    rows = args.ref_rows
    sec, threads = cpu_oracle_sample(N, k, cfg["group"], 1, rows, max(1, args.steps))
    value = alg_bytes(N, k) * (rows / N) / sec / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128, long double accumulation)",
            "data": "synthetic", "config": workload(cfg, k),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                             "sample": f"{rows} of {N} rows of Y = R X (k={k}), rows regenerated from the seed"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def workload(cfg, k):
    store = "complex128" if ES == 16.0 else "complex64-stored (FP64 arithmetic, complex128 vectors)"
    return {"workload": f"BASELINE.json config {cfg['id']}: TDA Hermitian N={cfg['N']} {store}, packed lower "
                        f"triangle {ES * cfg['N'] * (cfg['N'] + 1) / 2 / 1e9:.2f} GB, bse_apply k={k}",
            "N": cfg["N"], "k": k, "sigma": 0.0, "seed": 1, "storage": "c128" if ES == 16.0 else "c64",
            "l2": "operand larger than L2 (no flush needed)" if cfg["N"] >= 8192 else "operand L2-resident"}


def run_cuda(args, cfg):
    import torch
    import paper_2504_10096_b200 as b

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    N, k = cfg["N"], args.k

    storage = b.STORE_C128 if ES == 16.0 else b.STORE_C64
    shard = bool(args.shard)                                   # with one rank: the one-slice case of the same code path
    if shard:
        # ONE operand, its tile stream split over the ranks; each apply = local kernel + one all-reduce
        h = b.ShardedBse.synthetic(b.MODE_TDA, N, 1, 0.0, cfg["group"], storage=storage)
        tiles = None
    else:
        tiles = b.bse_fill_synthetic(N, b.MATRIX_R, 1, 0.0, cfg["group"], storage=storage)   # one operand per replica
        h = b.Bse(b.MODE_TDA, N, tiles, storage=storage)
    jobs = 1 if shard else world                                # independent operands in flight
    # FP64 tensor peak by the library's own DMMA probe, taken now at an unthrottled clock (burst figure, as hbm_gbs is);
    # `python bench.py --peaks` also measures it over seconds: the DMMA stream alone does not reach the power cap
    fp64_peak = b.selftest_peak(b.PEAK_DMMA, 8, 8)[0]
    Xh = torch.from_numpy(np.ascontiguousarray(gen.block_X(N, max(k, 8), 1001).T)).pin_memory()
    X = Xh[:k].cuda()
    Y = torch.empty_like(X)
    torch.cuda.synchronize()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: K applies
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    t_wait = time.time()
    if shard:
        # every apply contains a collective: all ranks must issue the same number of them, so no rank-local stop rule
        for _ in range(max(20, int(1.5e3 / max(1.0, alg_bytes(N, k) / world / 6.5e9)))):
            h.apply(X, Y)
        torch.cuda.synchronize()
    while not shard and not sampler.rows and time.time() - t_wait < 5.0:      # nvidia-smi takes a moment to start
        h.apply(X, Y)
        torch.cuda.synchronize()
    n_before = len(sampler.rows)
    l0 = b.launch_count()
    ms = time_steps(lambda: h.apply(X, Y), args.steps, args.warmup)
    launches = (b.launch_count() - l0) * args.steps // (args.steps + args.warmup)
    t_wait = time.time()
    if shard:
        for _ in range(max(20, int(1.5e3 / max(1.0, alg_bytes(N, k) / world / 6.5e9)))):     # ~1.5 s of the same load
            h.apply(X, Y)
        torch.cuda.synchronize()
    while not shard and len(sampler.rows) < n_before + 5 and time.time() - t_wait < 3.0:   # same load until >= 5 samples
        h.apply(X, Y)
        torch.cuda.synchronize()
    sampler.rows = sampler.rows[n_before:] if len(sampler.rows) > n_before else sampler.rows
    clocks = sampler.stop()
    barrier()
    ms = max_over_ranks(ms, dist, "cuda")
    value = jobs * alg_bytes(N, k) / (ms * 1e-3) / 1e9

    # ---- end to end through the host entry point (pinned host X and Y, copies inside the timed region)
    Xk = Xh[:k].numpy()
    Yk = torch.empty((k, N), dtype=torch.complex128).pin_memory().numpy()
    if shard:
        Xp, Yp = Xh[:k], torch.empty((k, N), dtype=torch.complex128).pin_memory()

        def host_step():                                        # pinned host X -> device, sharded apply, Y -> pinned host
            X.copy_(Xp, non_blocking=True)
            h.apply(X, Y)
            Yp.copy_(Y, non_blocking=True)
            torch.cuda.synchronize()
    else:
        def host_step():
            h.apply_host(Xk, Yk)
    for _ in range(2):
        host_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        host_step()
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / args.steps
    e2e_ms = max_over_ranks(e2e_ms, dist, "cuda")
    if dist is not None:
        barrier()
        dist.destroy_process_group()
        dist = None
    if rank != 0:
        return

    peak, peak_src = measured_peaks()
    achieved = alg_bytes(N, k) / (ms * 1e-3) / 1e9
    if shard:                                                   # per GPU: 1 / world of the tiles, the whole X and Y
        achieved = ((alg_bytes(N, k) - 32.0 * N * k) / world + 32.0 * N * k) / (ms * 1e-3) / 1e9
    traffic, traffic_src = None, None
    try:
        import csv
        # QUOTED from the committed ncu capture of the same kernel and workload (profiles/r2_apply_traffic.csv names the
        # capture); null when no capture of this workload exists -- it is not measured by the run that prints it
        with open(os.path.join(ROOT, "profiles", "r2_apply_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == f"N{N}_k{k}" + ("" if ES == 16.0 else "_c64"):
                    traffic = float(row["dram_bytes_per_launch"])
                    traffic_src = row["source"]
    except Exception:
        pass
    # north_star: roofline = min(bytes / HBM peak, flops / FP64 peak).  The FP64 figure is this repo's own DMMA
    # microbenchmark (bse_selftest_peak, `bench.py --peaks`): MEASURED_PEAKS.json has no FP64 entry.
    tflops = 8.0 * N * N * k / (ms * 1e-3) / 1e12 / (world if shard else 1)       # per GPU
    if 8.0 * N * N * k / (fp64_peak * 1e12) > alg_bytes(N, k) / (peak * 1e9):
        roof = {"bound": "tensor", "achieved": tflops, "peak": fp64_peak, "unit": "TFLOP/s", "frac": tflops / fp64_peak,
                "traffic": traffic, "peak_source": "bse_selftest_peak(BSE_PEAK_DMMA) measured in this run (burst; `python bench.py --peaks` has the sustained one)"}
    else:
        roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": peak_src}
    # 5 .. 8 columns: the kernel forms each complex product from three real ones (Role3M, apply_tiles.cuh), so the tensor
    # pipe executes 6 N^2 k flops for the 8 N^2 k algorithmic ones of SURVEY.md 8(d) that `achieved` counts.
    three_m = 5 <= k <= 8
    roof.update({"traffic_source": traffic_src, "kernel": "bse::apply_tiles_k1_kernel" if k == 1 else
                 ("bse::apply_tiles_kernel<16, Role3M>" if three_m else "bse::apply_tiles_kernel<16, Role4M>"),
                 "tflops_fp64": tflops, "tflops_fp64_executed": tflops * (0.75 if three_m else 1.0),
                 "fp64_peak_measured_tflops": fp64_peak, "GBps": achieved})
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong" if shard else "weak",
            "vs_baseline": None, "dtype": "f64 (complex128 on the FP64 tensor cores)", "data": "synthetic",
            "config": workload(cfg, k), "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": jobs * alg_bytes(N, k) / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": 16 * N * k, "d2h_bytes_per_step": 16 * N * k, "ms_per_step": e2e_ms},
            "roofline": roof}

    # ---- k sweep and Lanczos time-to-nev (the rest of BASELINE.json's metric), device-timed, outside `value`
    if shard:
        line["config"]["parallelism"] = f"tile stream sharded over {world} GPUs (contiguous tile rows, equal tile counts), " \
                                        "X replicated, one all-reduce of Y per apply"
    if not args.no_extras and ES == 16.0 and not shard:
        sweep = {}
        for kk in (1, 2, 4, 8):
            Xs, Ys = Xh[:kk].cuda(), torch.empty((kk, N), dtype=torch.complex128, device="cuda")
            m = time_steps(lambda: h.apply(Xs, Ys), max(3, args.steps // 2), 2)
            sweep[str(kk)] = {"ms": m, "GBps": alg_bytes(N, kk) / (m * 1e-3) / 1e9,
                              "tflops": 8.0 * N * N * kk / (m * 1e-3) / 1e12}
        line["apply_vs_k"] = sweep
        # Lanczos with quadrature: one k = 1 apply + three O(N) kernels per step
        dq = Xh[0].cuda()
        qsteps = 40
        h.lanczos_quadrature(dq, qsteps)                      # warm-up with the same step count: the timed call allocates nothing
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h.lanczos_quadrature(dq, qsteps)
        qsec = time.perf_counter() - t0
        line["lanczos_quadrature"] = {"steps": qsteps, "ms_per_step": qsec * 1e3 / qsteps,
                                      "GBps": alg_bytes(N, 1) * qsteps / qsec / 1e9}
        # Lanczos time-to-nev on the timed operand itself (BASELINE.json config 4: nev = 500, block k = 8, tol 1e-8)
        if cfg.get("id") == 4:
            t0 = time.perf_counter()
            res4 = h.solve(cfg["nev"], cfg["k"], tol=1e-8, seed=1, raise_on_error=False)
            line["lanczos_time_to_nev_config4"] = {
                "workload": f"config 4: TDA N={N} nev={cfg['nev']} k={cfg['k']} tol=1e-8", "seconds": time.perf_counter() - t0,
                "status": res4.status, "info": res4.info}
            del res4
        del h, tiles
        torch.cuda.empty_cache()
        # complex64-stored operand: same N, half the stored bytes, FP64 arithmetic.
        # Bytes are the complex64 store's; from k = 3 on the bound is the FP64 pipe, not HBM (ridge at 8 N^2 k / 37.1 TF).
        t64 = b.bse_fill_synthetic(N, b.MATRIX_R, 1, 0.0, cfg["group"], storage=b.STORE_C64)
        h64 = b.Bse(b.MODE_TDA, N, t64, storage=b.STORE_C64)
        sweep64 = {}
        for kk in (1, 2, 4, 8):
            Xs, Ys = Xh[:kk].cuda(), torch.empty((kk, N), dtype=torch.complex128, device="cuda")
            m = time_steps(lambda: h64.apply(Xs, Ys), max(3, args.steps // 2), 2)
            by = 8.0 * N * (N + 1) / 2 + 32.0 * N * kk
            sweep64[str(kk)] = {"ms": m, "GBps": by / (m * 1e-3) / 1e9, "tflops": 8.0 * N * N * kk / (m * 1e-3) / 1e12}
        line["apply_vs_k_c64_store"] = sweep64
        del h64, t64
        torch.cuda.empty_cache()
        c2 = gen.CONFIGS[2]
        h2 = b.Bse(b.MODE_TDA, c2["N"], b.bse_fill_synthetic(c2["N"], b.MATRIX_R, 1, 0.0, c2["group"]))
        # BASELINE.json config 2's k sweep (k > 8 is processed in groups of 8 columns, one pass over the operand each)
        sweep2 = {}
        X2 = torch.randn(64, c2["N"], dtype=torch.complex128, device="cuda")
        for kk in (1, 2, 4, 8, 16, 32, 64):
            Xs, Ys = X2[:kk], torch.empty((kk, c2["N"]), dtype=torch.complex128, device="cuda")
            m = time_steps(lambda: h2.apply(Xs, Ys), max(3, args.steps // 2), 2)
            sweep2[str(kk)] = {"ms": m, "GBps": alg_bytes(c2["N"], kk) / (m * 1e-3) / 1e9,
                               "tflops": 8.0 * c2["N"] ** 2 * kk / (m * 1e-3) / 1e12}
        line["apply_vs_k_config2"] = sweep2
        del X2
        t0 = time.perf_counter()
        res = h2.solve(c2["nev"], c2["k"], tol=1e-8, seed=1, raise_on_error=False)
        line["lanczos_time_to_nev"] = {"workload": f"config 2: TDA N={c2['N']} nev={c2['nev']} k={c2['k']} tol=1e-8",
                                       "seconds": time.perf_counter() - t0, "status": res.status, "info": res.info}
        del h2
        torch.cuda.empty_cache()
        # full-mode Lanczos with quadrature (PAPER.md:65 on Eq. 1) at config 3's size: per step two half applies with
        # k = 1, each streaming R and C once (4 tile passes of 8.59 GB)
        c3 = gen.CONFIGS[3]
        N3 = c3["N"]
        r3 = b.bse_fill_synthetic(N3, b.MATRIX_R, 1, 1.0, c3["group"])
        c3t = b.bse_fill_synthetic(N3, b.MATRIX_C, 1, 0.0, c3["group"])
        h3 = b.Bse(b.MODE_FULL, N3, r3, c3t)
        X3 = torch.randn(8, N3, dtype=torch.complex128, device="cuda")
        d3 = X3[0].contiguous()
        h3.lanczos_quadrature(d3, qsteps)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h3.lanczos_quadrature(d3, qsteps)
        qsec = time.perf_counter() - t0
        line["lanczos_quadrature_full"] = {"workload": f"config 3 operator: full N={N3}, sigma=1", "steps": qsteps,
                                           "ms_per_step": qsec * 1e3 / qsteps,
                                           "GBps": 4 * alg_bytes(N3, 1) * qsteps / qsec / 1e9}

        # full-mode half apply P(X) = R X + C conj(X) vs k: complex store (R and C passes) and the
        # real-form store of Eq. (3) (S = R + C, D = R - C; RoleReal in apply_tiles.cuh).  Bytes: both stores once + X, Y.
        def half_sweep(hh):
            out = {}
            for kk in (1, 4, 8):
                Xs = X3[:kk].contiguous()
                Ys = torch.empty_like(Xs)
                m = time_steps(lambda: hh.apply_half(Xs, 1, Ys), max(3, args.steps // 2), 2)
                by = 2 * 16.0 * N3 * (N3 + 1) / 2 + 32.0 * N3 * kk
                out[str(kk)] = {"ms": m, "GBps": by / (m * 1e-3) / 1e9}
            return out
        line["half_apply_vs_k_config3"] = half_sweep(h3)
        del h3
        b.bse_to_real_form(r3, c3t, N3)
        h3 = b.Bse(b.MODE_FULL, N3, r3, c3t, storage=b.STORE_REAL_FORM)
        line["half_apply_vs_k_config3_real_form"] = half_sweep(h3)
        t0 = time.perf_counter()
        res = h3.solve(c3["nev"], 8, tol=1e-8, seed=1, raise_on_error=False)
        line["lanczos_time_to_nev_config3"] = {
            "workload": f"config 3: full N={N3} nev={c3['nev']} k=8 tol=1e-8, real-form store", "seconds": time.perf_counter() - t0,
            "status": res.status, "info": res.info}
        del h3, r3, c3t
        torch.cuda.empty_cache()
        # the paper's direct route (section 2.1) on the device at config 1's size: every positive eigenpair of the 4096 x 4096 operator
        c1 = gen.CONFIGS[1]
        h1 = b.Bse(b.MODE_FULL, c1["N"], b.bse_fill_synthetic(c1["N"], b.MATRIX_R, 1, c1["sigma"], c1["group"]),
                   b.bse_fill_synthetic(c1["N"], b.MATRIX_C, 1, 0.0, c1["group"]))
        h1.solve_direct(4, vectors=False)                       # warm-up
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        om1, _, sec1 = h1.solve_direct(c1["N"])
        torch.cuda.synchronize()
        line["direct_route_config1"] = {"workload": f"config 1 operator: full N={c1['N']}, all {c1['N']} positive eigenpairs (bse_solve_direct)",
                                        "seconds": time.perf_counter() - t0, "stage_seconds": sec1, "omega_first": float(om1[0])}
        del h1

    # ---- CPU baseline: the oracle on this box's host cores, bounded sample
    if not args.no_cpu_baseline:
        sec, threads = cpu_oracle_sample(N, k, cfg["group"], 1, args.ref_rows, 3)
        # the verification oracle as it stands (dense row-major triple loop, x87 long-double accumulation, no SIMD, no use of
        # the Hermitian structure): a reported baseline, NOT a performance baseline -- a tuned CPU code would be far faster
        line["cpu_baseline"] = {"value": alg_bytes(N, k) * (args.ref_rows / N) / sec / 1e9, "unit": UNIT,
                                "cores": threads, "kind": "oracle",
                                "note": "verification oracle (long-double triple loop), not a tuned CPU implementation",
                                "sample": f"{args.ref_rows} of {N} rows of Y = R X (k={k}), 3 repetitions"}
    print(json.dumps(line))


def run_solve(spec):
    """`--solve CFG:K[:NCV[:STORE]]` -- time-to-nev of one bse_solve alone (the second half of BASELINE.json's metric), on
    the device-generated synthetic operator of BASELINE.json config CFG (2, 3 or 4; or MODE@N@NEV), block size K, basis size NCV (0 =
    default), STORE in {c128, c64, real, real64} (real*: the real-form store of DESIGN.md 5.5, full mode only).  Prints
    one JSON line; profiles/r2_solve.md's rows are runs of this command."""
    import torch
    import paper_2504_10096_b200 as b
    parts = spec.split(":")
    k = int(parts[1])
    ncv = int(parts[2]) if len(parts) > 2 and parts[2] else 0
    store = parts[3] if len(parts) > 3 and parts[3] else "c128"
    variant = {"shao": 0, "gruning": 1}[parts[4]] if len(parts) > 4 else 0      # bse_solve_variant
    if "@" in parts[0]:
        # MODE@N@NEV: the same generator at another size, e.g. the paper's N = 10368 / 36288 / 103680 with nev = 100
        # (PAPER.md:115-122, 180); sigma = 1 in full mode, group 16
        mode, n_, nev_ = parts[0].split("@")
        cid, cfg = parts[0], dict(mode=mode, N=int(n_), group=16, nev=int(nev_), sigma=1.0 if mode == "full" else 0.0)
    else:
        cid = int(parts[0])
        cfg = gen.CONFIGS[cid]
    N, full = cfg["N"], cfg["mode"] == "full"
    base = b.STORE_C64 if store in ("c64", "real64") else b.STORE_C128
    torch.cuda.set_device(0)
    rt = b.bse_fill_synthetic(N, b.MATRIX_R, 1, cfg["sigma"], cfg["group"], storage=base)
    ct = b.bse_fill_synthetic(N, b.MATRIX_C, 1, 0.0, cfg["group"], storage=base) if full else None
    storage = base
    if store.startswith("real"):
        if not full:
            raise SystemExit("the real-form store is a full-mode format")
        b.bse_to_real_form(rt, ct, N, storage=base)
        storage = b.STORE_REAL_FORM if base == b.STORE_C128 else b.STORE_REAL_FORM_C64
    h = b.Bse(b.MODE_FULL if full else b.MODE_TDA, N, rt, ct, storage=storage)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = h.solve(cfg["nev"], k, ncv=ncv, tol=1e-8, seed=1, raise_on_error=False, variant=variant)
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    print(json.dumps({"solve": {"workload": f"config {cid}: {cfg['mode']} N={N} nev={cfg['nev']} k={k} tol=1e-8 sigma={cfg['sigma']}",
                                "store": store, "variant": ["shao", "gruning"][variant], "seconds": sec, "status": res.status, "info": res.info,
                                "omega_first": float(res.omega[0]), "omega_last": float(res.omega[-1]),
                                "max_residual_estimate": float(res.resid.max())}}))


def run_direct(spec):
    """`--direct N[:NEV[:STORE]]` -- bse_solve_direct (the diagonalisation scheme of PAPER.md section 2.1 on the device) on the
    synthetic full-mode operator of BASELINE.json's generator at size N (sigma = 1, seed 1), NEV eigenpairs (default: all N,
    the direct route's use case; 0 = eigenvalues only).  Stage seconds from the library, wall time sync to sync, and the
    flop / byte counts of the stages.  One JSON line (profiles/r2_direct.md)."""
    import torch
    import paper_2504_10096_b200 as b
    parts = spec.split(":")
    N = int(parts[0])
    nev = int(parts[1]) if len(parts) > 1 and parts[1] else N
    store = parts[2] if len(parts) > 2 else "c128"
    torch.cuda.set_device(0)
    rt = b.bse_fill_synthetic(N, b.MATRIX_R, 1, 1.0, 16)
    ct = b.bse_fill_synthetic(N, b.MATRIX_C, 1, 0.0, 16)
    storage = b.STORE_C128
    if store == "real":
        b.bse_to_real_form(rt, ct, N)
        storage = b.STORE_REAL_FORM
    h = b.Bse(b.MODE_FULL, N, rt, ct, storage=storage)
    h.solve_direct(min(4, N), vectors=False) if N <= 2048 else None          # warm-up (module load, attributes) at small sizes
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    om, vec, sec = h.solve_direct(max(nev, 1), vectors=nev > 0)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    n = 2 * N
    out = {"workload": f"full N={N} (operator {n} x {n}) sigma=1.0 seed=1, nev={nev}", "store": store, "seconds_wall": wall,
           "seconds": sec, "omega_first": float(om[0]), "omega_last": float(om[-1]),
           "cholesky_tflops": (n ** 3 / 3) / max(sec["cholesky"], 1e-9) / 1e12,
           "w_tflops": 2.0 * n ** 3 / max(sec["w"], 1e-9) / 1e12,
           "tridiag_GBps": 8.0 / 3.0 * n ** 3 / max(sec["tridiag"], 1e-9) / 1e9}      # lower triangle read + written once per step
    if nev > 0:
        V = vec[: min(nev, 64)]
        HV = h.apply(V)
        w = torch.from_numpy(om[: V.shape[0]]).cuda()[:, None]
        out["max_residual_first_64"] = float((torch.linalg.vector_norm(HV - V * w, dim=1) / torch.linalg.vector_norm(V, dim=1)).max())
    print(json.dumps({"direct": out}))


def measure_peaks(b, sustained_s: float = 0.0):
    """The library's own microbenchmarks (bse_selftest_peak): burst figures from one timed launch each; with
    sustained_s > 0 also the rate of back-to-back launches over that many seconds (power cap reached)."""
    import torch
    out = {}

    def sustained(what, p1, p2, buf=None):
        t0, acc, n = time.perf_counter(), [], 0
        while time.perf_counter() - t0 < sustained_s:
            acc.append(b.selftest_peak(what, p1, p2, buf)[0]); n += 1
        tail = acc[len(acc) // 2:]
        return float(np.mean(tail)) if tail else None

    out["dmma_tflops"] = b.selftest_peak(b.PEAK_DMMA, 8, 8)[0]
    out["dmma_with_dadd_mix_tflops"] = b.selftest_peak(b.PEAK_DMMA, 8, -1)[0]
    out["dfma_tflops"] = b.selftest_peak(b.PEAK_DFMA, 32, 0)[0]
    buf = torch.empty(8 << 30, dtype=torch.uint8, device="cuda")
    buf.zero_()
    out["bulk_read_GBps"] = b.selftest_peak(b.PEAK_BULK_READ, 65536, 3, buf)[0]
    out["bulk_read_smem_readback_GBps"] = b.selftest_peak(b.PEAK_BULK_READ_SMEM, 65536, 3, buf)[0]
    small = torch.zeros(1536 * 1024, dtype=torch.float64, device="cuda")
    out["red_f64_Gops"] = b.selftest_peak(b.PEAK_RED, 0, 0, small)[0]
    if sustained_s > 0:
        out["dmma_tflops_sustained"] = sustained(b.PEAK_DMMA, 32, 8)
        out["dmma_with_dadd_mix_tflops_sustained"] = sustained(b.PEAK_DMMA, 32, -1)
        out["bulk_read_GBps_sustained"] = sustained(b.PEAK_BULK_READ, 65536, 3, buf)
        out["sustained_seconds_each"] = sustained_s
    del buf, small
    torch.cuda.empty_cache()
    return out


def run_peaks(args):
    """`--peaks`: one JSON line with the roofline denominators measured by the library itself (profiles/r2_peaks.md)."""
    import torch
    import paper_2504_10096_b200 as b
    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    sampler.start()
    out = measure_peaks(b, sustained_s=2.0)
    out["clocks"] = sampler.stop()
    hbm, src = measured_peaks()
    out["hbm_copy_GBps_driver"] = hbm
    print(json.dumps({"peaks": out}))


def run_dense(spec):
    """`--dense M:K[:L]`: the dense basis kernels at the shapes of a solve with basis width M, block K and rotation width L
    (default 3M/4) on N = 98304 rows (config 4): Gram (a5), skinny update (a6), Ritz rotation (a9), and one bse_orth call.
    CUDA events on the launch stream, 3 warm-ups, 10 timed launches each.  One JSON line (profiles/r2_dense_kernels.md)."""
    import torch
    import paper_2504_10096_b200 as b
    parts = [int(x) for x in spec.split(":")]
    m, k = parts[0], parts[1]
    l = parts[2] if len(parts) > 2 else (3 * m) // 4
    N = 98304
    torch.cuda.set_device(0)
    tiles = torch.zeros(b.bse_layout(1024)[2], dtype=torch.uint8, device="cuda")      # the dense kernels never touch the operator
    h = b.Bse(b.MODE_TDA, N, tiles)                                                     # (handle with N rows; tiles unused)
    V = torch.randn(m, N, dtype=torch.complex128, device="cuda") / np.sqrt(2 * N)
    W = torch.randn(k, N, dtype=torch.complex128, device="cuda")
    hbm, _ = measured_peaks()
    fp64 = b.selftest_peak(b.PEAK_DMMA, 8, 8)[0]
    out = {"N": N, "m": m, "k": k, "l": l, "fp64_peak_tflops": fp64, "hbm_peak_GBps": hbm}
    ms = time_steps(lambda: h.gram(V, W), 10, 3)
    by = 16.0 * N * (m + k)
    out["gram"] = {"ms": ms, "GBps": by / ms / 1e6, "frac_hbm": by / ms / 1e6 / hbm, "tflops": 8.0 * N * m * k / ms / 1e9}
    S = torch.randn(k, m, dtype=torch.complex128, device="cuda")
    ms = time_steps(lambda: h.update(V, S, W, -1.0, 1.0), 10, 3)
    by = 16.0 * N * (m + 2 * k)
    out["update"] = {"ms": ms, "GBps": by / ms / 1e6, "frac_hbm": by / ms / 1e6 / hbm}
    Sl = torch.randn(l, m, dtype=torch.complex128, device="cuda") / np.sqrt(m)
    Cout = torch.empty(l, N, dtype=torch.complex128, device="cuda")
    ms = time_steps(lambda: h.update(V, Sl, Cout), 5, 2)
    out["rotation"] = {"ms": ms, "tflops": 8.0 * N * m * l / ms / 1e9, "frac_fp64": 8.0 * N * m * l / ms / 1e9 / fp64}
    Q, _ = torch.linalg.qr(V[:min(m, 256)].T.contiguous())                              # orthonormal basis of the orth timing
    Vq = Q.T.contiguous()
    W0 = W.clone()

    def orth():
        W.copy_(W0)
        h.orth(Vq, W)
    ms = time_steps(orth, 10, 3)
    out["orth_call_m%d" % Vq.shape[0]] = {"ms": ms}
    print(json.dumps({"dense": out}))


def run_slices(args, cfg):
    """`--slices G` -- the G partial handles of a G-way partition of the timed operand, run ONE AFTER
    ANOTHER on this GPU: per-slice apply time (what each of G GPUs would spend in its local kernel, before the all-reduce
    of 16 N k bytes).  One JSON line; no multi-GPU claim."""
    import torch
    import paper_2504_10096_b200 as b
    torch.cuda.set_device(0)
    N, k = cfg["N"], args.k
    storage = b.STORE_C128 if ES == 16.0 else b.STORE_C64
    tiles = b.bse_fill_synthetic(N, b.MATRIX_R, 1, 0.0, cfg["group"], storage=storage)
    per = b.bse_layout(N, storage)[2] // b.bse_layout(N, storage)[1]
    X = torch.randn(k, N, dtype=torch.complex128, device="cuda")
    Y = torch.empty_like(X)
    out = {}
    for G in sorted({1, args.slices}):
        ms = []
        for r in range(G):
            rb, re, ft, n, by = b.bse_shard_layout(N, G, r, storage)
            h = b.Bse(b.MODE_TDA, N, tiles[ft * per: ft * per + max(by, 1)], storage=storage, rows=(rb, re))
            ms.append(time_steps(lambda: h.apply(X, Y), args.steps, args.warmup))
        out[str(G)] = {"ms_per_slice": ms, "max_ms": max(ms), "sum_ms": sum(ms)}
    whole = out["1"]["max_ms"]
    print(json.dumps({"slices": {"workload": workload(cfg, k), "per_partition": out,
                                 "balance": whole / (args.slices * out[str(args.slices)]["max_ms"])}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index (TDA ones: 0, 2, 4)")
    ap.add_argument("--k", type=int, default=4)
    ap.add_argument("--storage", default="c128", choices=["c128", "c64"],
                    help="c64: complex64-stored operand (SURVEY.md 8(f1)); the extras run for the default only")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1 GPUs: shard ONE operand's tile stream over the ranks (strong scaling) instead of replicas")
    ap.add_argument("--ref-rows", type=int, default=1024)
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--solve", default=None, metavar="CFG:K[:NCV[:STORE[:VARIANT]]]",
                    help="time one bse_solve alone (see run_solve) instead of the apply benchmark")
    ap.add_argument("--peaks", action="store_true", help="measure the roofline denominators with the library's microbenchmarks")
    ap.add_argument("--dense", default=None, metavar="M:K[:L]", help="time the dense basis kernels at config-4 shapes")
    ap.add_argument("--direct", default=None, metavar="N[:NEV[:STORE]]", help="time bse_solve_direct (PAPER.md section 2.1 on the device)")
    ap.add_argument("--slices", type=int, default=0, metavar="G",
                    help="time the G partial handles of a G-way partition one after another on this GPU (see run_slices)")
    args = ap.parse_args()
    if args.solve:
        run_solve(args.solve)
        return
    if args.direct:
        run_direct(args.direct)
        return
    if args.peaks:
        run_peaks(args)
        return
    if args.dense:
        run_dense(args.dense)
        return
    args.warmup = max(args.warmup, 3)
    global ES
    ES = 16.0 if args.storage == "c128" else 8.0
    cfg = dict(gen.CONFIGS[args.config], id=args.config)
    if cfg["mode"] != "tda":
        raise SystemExit("bench.py times the TDA apply; full-mode configs are parity-test cases")
    if args.slices > 0:
        run_slices(args, cfg)
    elif args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_cuda(args, cfg)


if __name__ == "__main__":
    main()
