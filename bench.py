#!/usr/bin/env python
"""bench.py -- the hot path of arXiv 1311.2719 on B200: conjugate-gradient fermion solver.

One "step" = one call of the paper's congrad: the whole hot path of SURVEY.md
8(a) -- init (S6), then per iteration Dslash-1 + alpha (S1,S2), Dslash-2 fused with the x/r
updates and |r|^2 (S3), the convergence scalar (S4), the p-update (S5), and the true-residual
check (S7) -- on BASELINE.json config 3 (32^4 staggered, Haar links, m = 0.01, tol 1e-10), the
configuration the north-star target is quoted on.  `value` = algorithmic HBM bytes of the solve
(2832 B per site and iteration + init + final check) / time-to-solution, summed
over ranks; `ms_per_step` is the CG time-to-solution.  `roofline` is the plain staggered Dslash
kernel (1248 B per output site) timed with CUDA events on the library's stream.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5]

N > 1 (torchrun): replicas only -- every rank solves its own right-hand side on the same gauge
field, no data-path collective; scaling = weak.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1311_2719_b200 import synth  # noqa: E402  (input generators only)

STAG_DSLASH_BYTES = 1248   # per output site: 8 links x 144 B + 48 B in + 48 B out
STAG_DSLASH_FLOPS = 570
WILSON_DSLASH_BYTES = 1536
WILSON_DSLASH_FLOPS = 1320
NOMINAL_HBM_GBS = 8000.0
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent


def cg_bytes(cfg, iters: int, recon: int = 18, updates: int = -1) -> float:
    """Algorithmic HBM bytes of one solve; links cost 8 x recon x 8 B per site.
    updates >= 0: the mixed-precision solver (fp32 iterations + that many fp64 reliable updates)."""
    v = synth.volume(cfg["dims"])
    links = 8 * recon * 8                                 # 1152 B (all nine entries) or 768 B (two rows)
    if cfg["fermion"] == "staggered":
        vh, vec = v // 2, 48
        per_iter = 2 * links + 11 * vec                   # 2832 B / site / iteration at recon 18
        fixed = 4 * vec + (links + 2 * vec) + (links + 4 * vec)  # init + D_oe x + fused residual
        if updates >= 0:
            per_iter = per_iter // 2                      # fp32 links and vectors: 1416 / 1032 B
            # reliable update: x += xs (24 + 2*48), D_oe x (links + 2*48), D_eo + r (links + 3*48 + 24), p-update (3*24)
            per_update = (24 + 2 * vec) + (links + 2 * vec) + (links + 3 * vec + 24) + 72
            fixed = (vec + 3 * 24 + vec) + (24 + 2 * vec) + (links + 2 * vec) + (links + 4 * vec) + updates * per_update
        return float(vh) * (per_iter * iters + fixed)
    vec = 192
    per_iter = 2 * links + 11 * vec                       # two full-lattice hops + 11 vector passes
    fixed = 4 * vec + (links + 2 * vec) + (links + 3 * vec)
    return float(v) * (per_iter * iters + fixed)


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the roofline kernel, from the committed
    ncu --set full capture (profiles/traffic.csv); None if that kernel/workload was not captured."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for row in open(path).read().splitlines()[1:]:
            f = row.split(",")
            if f[0] == key:
                return int(f[1]) + int(f[2])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, val in zip(names, f[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_arm(cfg, u, b, steps, warmup, target_seconds=6.0):
    """The oracle as it stands on the host cores: each step = `n_it` CG iterations (tol = 0)."""
    import oracle
    f = 0 if cfg["fermion"] == "staggered" else 1
    t0 = time.perf_counter()
    oracle.cg(cfg["dims"], f, u, cfg["param"], 0.0, 1, b)
    t1 = time.perf_counter() - t0
    n_it = max(1, int(target_seconds / max(t1 / 2.0, 1e-6)))   # a 1-iteration call applies A twice (loop + check)
    n_it = min(n_it, 200)
    for _ in range(warmup):
        oracle.cg(cfg["dims"], f, u, cfg["param"], 0.0, 1, b)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        oracle.cg(cfg["dims"], f, u, cfg["param"], 0.0, n_it, b)
        times.append(time.perf_counter() - t0)
    sec = sum(times) / len(times)
    return {"value": cg_bytes(cfg, n_it) / sec / 1e9, "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": "%d CG iterations (tol=0) of the %s solve per step, %d steps, %.2f s/step"
                      % (n_it, cfg["name"], steps, sec), "ms_per_step": sec * 1e3, "iters_per_step": n_it}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--cg-mode", default="graph", choices=["sync", "async", "graph"])
    ap.add_argument("--check-every", type=int, default=8)
    ap.add_argument("--dslash-reps", type=int, default=200)
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12],
                    help="stored reals per link: 18 = all nine entries (the roofline workload), 12 = two rows")
    ap.add_argument("--precision", default="f64", choices=["f64", "mixed"],
                    help="f64 = the fp64 conjugate gradient (the headline); mixed = fp32 iterations + fp64 reliable updates")
    ap.add_argument("--delta", type=float, default=0.1, help="reliable-update threshold of --precision mixed")
    ap.add_argument("--no-variants", action="store_true", help="skip the extra recon-12 / mixed-precision solves")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    cfg = synth.config(args.config)
    workload = "%s: %s %s, %s links, %s=%g, tol=%g, fp64" % (
        cfg["name"], "x".join(map(str, cfg["dims"])), cfg["fermion"], cfg["links"],
        "mass" if cfg["fermion"] == "staggered" else "kappa", cfg["param"], cfg["tol"])
    metric = "CG solve effective HBM throughput (algorithmic bytes of Dslash + fused updates / time-to-solution)"

    # ------------------------------------------------------------------ reference arm = the oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        u = synth.gauge_field(cfg["dims"], cfg["links"], cfg["seed"])
        b = synth.source(cfg["dims"], cfg["fermion"], cfg["seed"])
        r = oracle_arm(cfg, u, b, max(1, args.steps), max(0, args.warmup), target_seconds=8.0)
        line = {"impl": "reference", "metric": metric, "value": r["value"], "unit": "GB/s", "n_gpus": 0,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload, "sample": r["sample"]},
                "cpu_baseline": {"value": r["value"], "unit": "GB/s", "cores": r["cores"], "kind": "oracle",
                                 "sample": r["sample"]},
                "e2e": {"value": r["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line))
        return 0

    # ------------------------------------------------------------------ our arm
    import torch
    from paper_1311_2719_b200 import lqcd
    from paper_1311_2719_b200.ranks import Ranks

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path is the only path")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    ranks = Ranks(backend="nccl", device=device)
    barrier, max_over_ranks, sum_over_ranks = ranks.barrier, ranks.max, ranks.sum

    f = lqcd.STAGGERED if cfg["fermion"] == "staggered" else lqcd.WILSON
    u = synth.gauge_field(cfg["dims"], cfg["links"], cfg["seed"])
    b = synth.source(cfg["dims"], cfg["fermion"], ranks.rhs_seed(cfg["seed"]))   # one right-hand side per rank
    u_host = torch.from_numpy(u).pin_memory()
    b_host = torch.from_numpy(b).pin_memory()
    lat = lqcd.Lattice(cfg["dims"], f, device=device)
    lat.set_option(lqcd.OPT_CG_MODE, {"sync": lqcd.CG_SYNC, "async": lqcd.CG_ASYNC, "graph": lqcd.CG_GRAPH}[args.cg_mode])
    lat.set_option(lqcd.OPT_CG_CHECK_EVERY, args.check_every)
    lat.set_option(lqcd.OPT_RECONSTRUCT, args.recon)
    u_dev = u_host.to(device, non_blocking=True)
    b_dev = b_host.to(device, non_blocking=True)
    lat.load_gauge(u_dev)
    x_dev = lat.new_vector()
    maxiter = 100000
    v = synth.volume(cfg["dims"])
    sites_out = v // 2   # output sites of one parity Dslash

    mixed = args.precision == "mixed"
    if mixed and f != lqcd.STAGGERED:
        raise SystemExit("--precision mixed is built for the staggered configs")
    updates = -1

    def solve():
        """One step = one whole solve; returns (iters, reliable updates or -1, true residual, status)."""
        if mixed:
            _, it_, nu_, res_, st_ = lat.cg_solve_mixed(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev, delta=args.delta)
            return it_, nu_, res_, st_
        _, it_, res_, st_ = lat.cg_solve(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev)
        return it_, -1, res_, st_

    # warm-up
    iters = res = None
    for _ in range(max(args.warmup, 3)):
        iters, updates, res, status = solve()
    assert status == 0, "CG did not converge"

    # ---- timed region 1: K whole solves, device-resident inputs
    sampler = ClockSampler(local_rank) if rank == 0 else None
    launches0 = lat.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(lat.stream)
    for _ in range(args.steps):
        iters, updates, res, status = solve()
    e1.record(lat.stream)
    barrier()
    ms_solve = max_over_ranks(e0.elapsed_time(e1)) / args.steps
    launches = lat.kernel_launches() - launches0
    total_bytes = sum_over_ranks(cg_bytes(cfg, iters, args.recon, updates))
    value = total_bytes / (ms_solve * 1e-3) / 1e9

    # ---- timed region 2: the dominant kernel alone (plain Dslash), CUDA events on its stream.
    # Inputs (0.6 GB of links at cfg 3) exceed the 126 MB L2, parities alternate.
    if f == lqcd.STAGGERED:
        va, vb = lat.new_vector(), lat.new_vector()
        va.copy_(b_dev)
        dbytes, dflops = STAG_DSLASH_BYTES - 8 * 8 * (18 - args.recon), STAG_DSLASH_FLOPS
    else:
        va, vb = lat.new_vector(), lat.new_vector()
        va.copy_(b_dev)
        vb.zero_()
        dbytes, dflops = WILSON_DSLASH_BYTES - 8 * 8 * (18 - args.recon), WILSON_DSLASH_FLOPS
    for i in range(6):
        lat.dslash(1 - (i & 1), va if not (i & 1) else vb, vb if not (i & 1) else va)
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    d0.record(lat.stream)
    for i in range(args.dslash_reps):
        lat.dslash(1 - (i & 1), va if not (i & 1) else vb, vb if not (i & 1) else va)
    d1.record(lat.stream)
    barrier()
    us_dslash = max_over_ranks(d0.elapsed_time(d1)) * 1e3 / args.dslash_reps
    clocks = sampler.stop() if sampler else None
    peak, peak_src = hbm_peak()
    achieved = dbytes * sites_out / (us_dslash * 1e-6) / 1e9

    # ---- e2e: the paper's congrad with its data region, HOST buffers through the C-ABI
    e2e = None
    if not args.no_e2e:
        x_host = torch.empty(lat.vector_shape, dtype=torch.complex128).pin_memory()
        lat.set_option(lqcd.OPT_CONGRAD_PRECISION, 32 if mixed else 64)
        lat.congrad_host(u_host, cfg["param"], cfg["tol"], maxiter, b_host, x_host)   # warm
        n_e2e = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            _, it_e, res_e, st_e = lat.congrad_host(u_host, cfg["param"], cfg["tol"], maxiter, b_host, x_host)
        torch.cuda.synchronize()
        sec = max_over_ranks(time.perf_counter() - t0) / n_e2e
        e2e = {"value": sum_over_ranks(cg_bytes(cfg, it_e, args.recon, updates)) / sec / 1e9, "unit": "GB/s", "ms_per_step": sec * 1e3,
               "h2d_bytes_per_step": int(u_host.numel() * 16 + b_host.numel() * 16),
               "d2h_bytes_per_step": int(x_host.numel() * 16 + 128), "iters": it_e, "true_residual": res_e,
               "api": "lqcd_congrad_host (pinned host u, b -> x)"}

    # ---- the other solver variants on the same workload: time-to-solution only (one warm-up, one timed solve)
    variants = None
    if f == lqcd.STAGGERED and not args.no_variants:
        variants = {}
        for recon_v, prec_v in ((18, "f64"), (12, "f64"), (18, "mixed"), (12, "mixed")):
            if (recon_v, prec_v) == (args.recon, args.precision):
                continue
            lat.set_option(lqcd.OPT_RECONSTRUCT, recon_v)
            lat.load_gauge(u_dev)
            v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for rep in range(2):
                barrier()
                v0.record(lat.stream)
                if prec_v == "mixed":
                    _, it_v, nu_v, res_v, st_v = lat.cg_solve_mixed(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev,
                                                                    delta=args.delta)
                else:
                    _, it_v, res_v, st_v = lat.cg_solve(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev)
                    nu_v = -1
                v1.record(lat.stream)
                barrier()
            ms_v = max_over_ranks(v0.elapsed_time(v1))
            variants["%s_recon%d" % (prec_v, recon_v)] = {
                "time_to_solution_ms": ms_v, "iters": it_v, "reliable_updates": nu_v if nu_v >= 0 else None,
                "true_residual": res_v, "converged": st_v == 0,
                "GBps": sum_over_ranks(cg_bytes(cfg, it_v, recon_v, nu_v)) / (ms_v * 1e-3) / 1e9}
        lat.set_option(lqcd.OPT_RECONSTRUCT, args.recon)
        lat.load_gauge(u_dev)

    # ---- the oracle beside it (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r = oracle_arm(cfg, u, b, steps=2, warmup=0, target_seconds=6.0)
        cpu = {"value": r["value"], "unit": "GB/s", "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}

    if rank == 0:
        line = {
            "metric": metric, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_solve, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if not mixed else "f32 iterations + f64 reliable updates",
            "data": "synthetic",
            "config": {"workload": workload, "precision": args.precision, "reconstruct": args.recon, "cg_mode": args.cg_mode, "check_every": args.check_every,
                       "parallelism": "replicas x%d (independent right-hand sides)" % world,
                       "l2_policy": "inputs larger than L2 (%.0f MB of links per Dslash), no flush" % (v * 576 / 1e6)},
            "cg": {"time_to_solution_ms": ms_solve, "iters": iters, "reliable_updates": updates if mixed else None,
                   "true_residual": res,
                   "us_per_iteration": ms_solve * 1e3 / max(iters, 1)},
            "dslash": {"us_per_call": us_dslash, "GBps": achieved, "GFLOPs": dflops * sites_out / (us_dslash * 1e-6) / 1e9,
                       "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS, "reps": args.dslash_reps},
            "roofline": {"bound": "hbm", "kernel": "stag_dslash_kernel<SE_PLAIN>" if f == lqcd.STAGGERED else
                         "wilson_dslash_kernel<WE_PLAIN>", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "peak_source": peak_src, "traffic": None,
                         "bytes_per_site": dbytes, "sites_per_launch": sites_out},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "cpu_baseline": cpu, "variants": variants,
        }
        line["roofline"]["traffic"] = ncu_traffic("%s_dslash_plain%s" % (cfg["name"], "" if args.recon == 18 else "_recon12"))
        print(json.dumps(line))
    lat.close()
    ranks.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
