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

N > 1 (torchrun): by default replicas -- every rank solves its own right-hand side on the same gauge
field, no data-path collective; scaling = weak.  --parallelism slab: ONE system cut
into time-slabs, one per GPU (include/lqcd_slab.h: halo stores and sums through peer memory); scaling =
strong; not yet timed on more than one GPU.
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
L2_BYTES = 126e6           # B200 L2 (B200_PROFILING.md); the library's own rule reads cudaDevAttrL2CacheSize


def links_fit_l2(cfg, recon: int) -> bool:
    """The library's rule for the one-kernel loop (lqcd_load_gauge): the stored links take at most a third of the L2."""
    return synth.volume(cfg["dims"]) * 4 * (recon // 2) * 16 <= L2_BYTES / 3


def expected_cg_path(args, cfg) -> str:
    """Which iteration loop lqcd_cg_solve runs for these flags (LQCD_OPT_PERSISTENT = -1, automatic): the one
    cooperative kernel where the links fit the L2 -- staggered fp64 solves only, and never against an explicit
    --cg-mode sync -- else the host loop in the --cg-mode form.  ours_line checks it against lqcd_last_cg_path()."""
    if cfg["fermion"] == "staggered" and args.precision == "f64" and args.cg_mode != "sync" and links_fit_l2(cfg, args.recon):
        return "persistent"
    return "host_loop"


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
        rows = [row.split(",") for row in open(path).read().splitlines()[1:]]
        for want in ("r02_" + key, key):   # the newest capture of that kernel / workload
            for f in rows:
                if f[0] == want:
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


def workload_name(cfg):
    return "%s: %s %s, %s links, %s=%g, tol=%g, fp64" % (
        cfg["name"], "x".join(map(str, cfg["dims"])), cfg["fermion"], cfg["links"],
        "mass" if cfg["fermion"] == "staggered" else "kappa", cfg["param"], cfg["tol"])


def config_dict(args, cfg, world):
    """The `config` object of the JSON line: the same keys and values in our arm and in the reference arm
    (what the reference arm samples of the workload is said in its cpu_baseline.sample)."""
    link_mb = synth.volume(cfg["dims"]) * 4 * (args.recon // 2) * 16 / 1e6
    path = expected_cg_path(args, cfg)
    if path == "persistent":
        mode = "persistent: the loop is one cooperative kernel, exit test on the device (cg_mode %s / check_every %d not used)" % (
            args.cg_mode, args.check_every)
    else:
        mode = args.cg_mode
    if link_mb * 1e6 > L2_BYTES:
        l2 = "inputs larger than L2 (%.0f MB of links per Dslash against %.0f MB), no flush" % (link_mb, L2_BYTES / 1e6)
    elif path == "persistent":
        l2 = "L2-RESIDENT workload by design (%.1f MB of links fit the %.0f MB L2; no flush): the times are L2 times, not HBM times" % (
            link_mb, L2_BYTES / 1e6)
    else:
        l2 = "%.0f MB of links against %.0f MB of L2: partly L2-resident, no flush" % (link_mb, L2_BYTES / 1e6)
    return {"workload": workload_name(cfg), "precision": args.precision, "reconstruct": args.recon,
            "cg_mode": mode, "cg_path": path, "check_every": args.check_every if path == "host_loop" else None,
            "parallelism": "replicas x%d (independent right-hand sides)" % world,
            "l2_policy": l2}


def oracle_dslash_times(cfg, u, b, budget_s=4.0):
    """The oracle's hopping term alone (SURVEY 8(d) timing protocol; the paper's fmv/fmtv):
    microseconds per call on all host cores and on one thread, beside the GPU's dslash.us_per_call."""
    import oracle
    f = 0 if cfg["fermion"] == "staggered" else 1
    nbytes = (STAG_DSLASH_BYTES if f == 0 else WILSON_DSLASH_BYTES) * (synth.volume(cfg["dims"]) // 2)
    all_threads = oracle.num_threads()
    out = {"cores": all_threads}
    for label, nthr in (("all_cores", all_threads), ("one_thread", 1)):
        oracle.set_threads(nthr)
        try:
            t0 = time.perf_counter()
            oracle.dslash(cfg["dims"], f, u, 1, b)
            t1 = time.perf_counter() - t0
            reps = max(1, min(50, int(budget_s / 2 / max(t1, 1e-6))))
            t0 = time.perf_counter()
            for _ in range(reps):
                oracle.dslash(cfg["dims"], f, u, 1, b)
            sec = (time.perf_counter() - t0) / reps
        finally:
            oracle.set_threads(all_threads)
        out["us_per_call_" + label] = sec * 1e6
        out["GBps_" + label] = nbytes / sec / 1e9
        out["reps_" + label] = reps
    return out


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


def slab_group_variant(slab_mod, cfg, ug, bg, R, args, maxiter, mixed=False):
    """Time-to-solution of the R-slab decomposition with all slabs on this GPU (one warm-up + one timed solve);
    mixed = True: the mixed-precision slab solver (lqcd_slab_cg_solve_mixed_group)."""
    import torch
    grp = slab_mod.SlabGroup(cfg["dims"], R, recon=args.recon)
    try:
        grp.set_option(slab_mod.OPT_CHECK_EVERY, args.check_every)
        grp.load_gauge_from_global(ug)
        bs, xs = grp.scatter(bg), grp.new_vectors()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        st = grp.slabs[0].stream
        for rep in range(2):
            torch.cuda.synchronize()
            g0.record(st)
            if mixed:
                _, it_g, nu_g, res_g, st_g = grp.cg_solve_mixed(cfg["param"], cfg["tol"], maxiter, bs, xs, delta=args.delta)
            else:
                _, it_g, res_g, st_g = grp.cg_solve(cfg["param"], cfg["tol"], maxiter, bs, xs)
                nu_g = -1
            g1.record(st)
            torch.cuda.synchronize()
        ms_g = g0.elapsed_time(g1)
        return {"time_to_solution_ms": ms_g, "iters": it_g, "reliable_updates": nu_g if mixed else None,
                "true_residual": res_g, "converged": st_g == 0,
                "GBps": cg_bytes(cfg, it_g, args.recon, nu_g) / (ms_g * 1e-3) / 1e9}
    finally:
        grp.close()


def slab_strong_variant(args, cfg, ranks, device, maxiter):
    """One solve of cfg as N time-slabs, one per rank/GPU (collective: every rank calls it).  Returns a dict on every
    rank; an {"error": ...} dict on EVERY rank if anything fails on any rank.  Failure-safe by construction: after each
    phase that can fail locally the ranks agree (an all-reduce every rank reaches) whether to go on, the waits inside
    the solver are bounded (LQCD_ECOMM), so no rank is ever left in a collective its peers have abandoned."""
    import torch
    from paper_1311_2719_b200 import slab as sl
    rank, world = ranks.rank, ranks.world
    dims = cfg["dims"]
    if dims[3] % world or (dims[3] // world) % 2 or dims[3] // world < 2:   # the same verdict on every rank
        return {"error": "L3 = %d cannot be cut into %d even slabs" % (dims[3], world)}
    state = {"s": None, "why": ""}

    def agreed(step):
        """Run a local step; then every rank learns whether all of them succeeded."""
        bad = 0.0
        try:
            step()
        except Exception as exc:  # noqa: BLE001
            state["why"] = repr(exc)[:300]
            bad = 1.0
        return ranks.sum(bad) == 0

    def give_up(where):
        try:
            if state["s"] is not None:
                state["s"].close()
        except Exception:  # noqa: BLE001
            pass
        return {"error": "%s: %s" % (where, state["why"] or "a peer failed")}

    def create():
        ug = torch.from_numpy(synth.gauge_field(dims, cfg["links"], cfg["seed"]))
        bg = torch.from_numpy(synth.source(dims, cfg["fermion"], cfg["seed"]))
        s = sl.Slab(dims, rank, world, device=device)
        state["s"] = s
        s.set_option(sl.OPT_RECONSTRUCT, args.recon)
        s.set_option(sl.OPT_CHECK_EVERY, args.check_every)
        s.set_option(sl.OPT_TIMEOUT_MS, 10000)
        state["u"] = (sl.local_gauge(ug, dims, rank, world), sl.u3_below_from_global(ug, dims, rank, world))
        state["b"] = sl.local_vector(bg, dims, rank, world)

    if not agreed(create):
        return give_up("set-up")
    if not agreed(lambda: state["s"].connect_ipc()):   # itself collective and failure-safe (slab.py)
        return give_up("connect_ipc")
    s = state["s"]

    def load():
        s.load_gauge(state["u"][0].to(device), state["u"][1].to(device))
        state["bd"], state["xd"] = state["b"].to(device), s.new_vector()

    if not agreed(load):
        return give_up("load_gauge")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for rep in range(2):   # one warm-up, one timed

        def solve():
            e0.record(s.stream)
            state["res"] = s.cg_solve(cfg["param"], cfg["tol"], maxiter, state["bd"], state["xd"])
            e1.record(s.stream)
            torch.cuda.synchronize(device)

        ranks.barrier()
        if not agreed(solve):
            return give_up("cg_solve")
    _, it, res, st = state["res"]
    ms = ranks.max(e0.elapsed_time(e1))
    sh = dims[0] * dims[1] * dims[2] // 2
    out = {"time_to_solution_ms": ms, "iters": it, "true_residual": res, "converged": st == 0,
           "GBps": cg_bytes(cfg, it, args.recon) / (ms * 1e-3) / 1e9, "scaling": "strong",
           "nvlink_bytes_per_dslash_and_rank": 2 * sh * 48, "sync_points": s.sync_points(),
           "note": "one system, T = %d time-slices per GPU; first multi-GPU run of this path: check against the N = 1 solve" % (dims[3] // world)}
    try:
        s.close()
    except Exception:  # noqa: BLE001
        pass
    return out


def slab_arm(args, cfg, workload, metric, ranks, device):
    """--parallelism slab: ONE system on N GPUs, rank r owns time-slab r (strong scaling).  One process
    per GPU; the mailboxes are mapped across processes with CUDA IPC; every hot step -- hopping terms,
    halo stores into the neighbours' ghost faces, rank-ordered sums, the CG -- is in the CUDA library."""
    import torch
    from paper_1311_2719_b200 import slab as sl
    if cfg["fermion"] != "staggered":
        raise SystemExit("--parallelism slab is built for the staggered configs")
    rank, world = ranks.rank, ranks.world
    dims = cfg["dims"]
    ug = torch.from_numpy(synth.gauge_field(dims, cfg["links"], cfg["seed"]))      # every rank builds the global field,
    bg = torch.from_numpy(synth.source(dims, cfg["fermion"], cfg["seed"]))         # keeps its slab
    s = sl.Slab(dims, rank, world, device=device)
    s.set_option(sl.OPT_RECONSTRUCT, args.recon)
    s.set_option(sl.OPT_CHECK_EVERY, args.check_every)
    s.connect_ipc()
    u_local = sl.local_gauge(ug, dims, rank, world).pin_memory()
    u3_below = sl.u3_below_from_global(ug, dims, rank, world).pin_memory()
    b_host = sl.local_vector(bg, dims, rank, world).pin_memory()
    del ug, bg
    s.load_gauge(u_local.to(device), u3_below.to(device))
    b_dev, x_dev = b_host.to(device), s.new_vector()
    maxiter = 100000
    vh = synth.volume(dims) // 2
    for _ in range(max(args.warmup, 3)):
        _, iters, res, status = s.cg_solve(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev)
    assert status == 0, "CG did not converge"
    sampler = ClockSampler(ranks.local_rank) if rank == 0 else None
    launches0 = s.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ranks.barrier()
    e0.record(s.stream)
    for _ in range(args.steps):
        _, iters, res, status = s.cg_solve(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev)
    e1.record(s.stream)
    ranks.barrier()
    ms_solve = ranks.max(e0.elapsed_time(e1)) / args.steps
    launches = ranks.sum(s.kernel_launches() - launches0)
    value = cg_bytes(cfg, iters, args.recon) / (ms_solve * 1e-3) / 1e9            # the ONE global solve
    # the slab hopping term alone (face push + synchronisation point + Dslash per call)
    va, vb = s.new_vector(), s.new_vector()
    va.copy_(b_dev)
    for i in range(6):
        s.dslash(1 - (i & 1), va if not (i & 1) else vb, vb if not (i & 1) else va)
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ranks.barrier()
    d0.record(s.stream)
    for i in range(args.dslash_reps):
        s.dslash(1 - (i & 1), va if not (i & 1) else vb, vb if not (i & 1) else va)
    d1.record(s.stream)
    ranks.barrier()
    us_dslash = ranks.max(d0.elapsed_time(d1)) * 1e3 / args.dslash_reps
    clocks = sampler.stop() if sampler else None
    dbytes = STAG_DSLASH_BYTES - 8 * 8 * (18 - args.recon)
    achieved = dbytes * vh / (us_dslash * 1e-6) / 1e9                              # all ranks together
    peak, peak_src = hbm_peak()
    # e2e: this rank's slab of u and b from pinned host memory, x back, inside the timed region
    e2e = None
    if not args.no_e2e:
        x_host = torch.empty(s.vector_shape, dtype=torch.complex128).pin_memory()
        ranks.barrier()
        t0 = time.perf_counter()
        s.load_gauge(u_local.to(device, non_blocking=True), u3_below.to(device, non_blocking=True))
        bd = b_host.to(device, non_blocking=True)
        _, it_e, res_e, st_e = s.cg_solve(cfg["param"], cfg["tol"], maxiter, bd, x_dev)
        x_host.copy_(x_dev)
        torch.cuda.synchronize()
        sec = ranks.max(time.perf_counter() - t0)
        e2e = {"value": cg_bytes(cfg, it_e, args.recon) / sec / 1e9, "unit": "GB/s", "ms_per_step": sec * 1e3,
               "h2d_bytes_per_step": int(ranks.sum((u_local.numel() + u3_below.numel() + b_host.numel()) * 16)),
               "d2h_bytes_per_step": int(ranks.sum(x_host.numel() * 16 + 128)), "iters": it_e, "true_residual": res_e,
               "api": "slab.Slab.load_gauge + cg_solve (pinned host u_local, b_local -> x_local)"}
    if rank == 0:
        line = {
            "metric": metric, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_solve, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload, "precision": "f64", "reconstruct": args.recon, "cg_mode": "async",
                       "check_every": args.check_every,
                       "parallelism": "time-slabs x%d (one system; T = %d slices per GPU; peer-memory halo + sums)" % (world, dims[3] // world),
                       "l2_policy": "inputs larger than L2 (%.0f MB of links per Dslash and GPU), no flush" % (2 * vh * 576 / 1e6 / world)},
            "cg": {"time_to_solution_ms": ms_solve, "iters": iters, "true_residual": res,
                   "us_per_iteration": ms_solve * 1e3 / max(iters, 1), "sync_points": s.sync_points()},
            "dslash": {"us_per_call": us_dslash, "GBps": achieved, "GFLOPs": STAG_DSLASH_FLOPS * vh / (us_dslash * 1e-6) / 1e9,
                       "reps": args.dslash_reps, "note": "lqcd_slab_dslash: face push + synchronisation point + hopping term"},
            "roofline": {"bound": "hbm", "kernel": "stag_dslash_slab_kernel<SE_PLAIN> (+ face push, signal, wait)",
                         "achieved": achieved / world, "peak": peak, "unit": "GB/s", "frac": achieved / world / peak,
                         "peak_source": peak_src + "; achieved is per GPU", "traffic": None, "bytes_per_site": dbytes,
                         "sites_per_launch": vh // world},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "cpu_baseline": None, "variants": None,
        }
        print(json.dumps(line))
    s.close()
    ranks.close()
    return 0


def ours_line(args, cfg, metric, ranks, device, lqcd, torch, full=True, solver_variants=None):
    """Our arm on one config: returns the JSON line (a dict) on every rank.  full = False (--all-configs, and the
    `configs` entries of the default line): no oracle timing, no slab variants, and the other solvers on the same
    workload (two-row links, mixed precision; Wilson: the even-odd solve) only if solver_variants is set."""
    if solver_variants is None:
        solver_variants = full
    rank, world, local_rank = ranks.rank, ranks.world, ranks.local_rank
    barrier, max_over_ranks, sum_over_ranks = ranks.barrier, ranks.max, ranks.sum
    workload = workload_name(cfg)
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
    path_ran = {lqcd.PATH_HOST_LOOP: "host_loop", lqcd.PATH_PERSISTENT: "persistent"}.get(lat.last_cg_path(), "none")

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
    # lqcd_dslash_sweep enqueues the launches natively (odd parity first, ping-pong va -> vb -> va ...):
    # no Python between launches, so the small lattices are timed on the device too.
    lat.dslash_sweep(1, va, vb, 6)
    d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    d0.record(lat.stream)
    lat.dslash_sweep(1, va, vb, args.dslash_reps)
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
    if f == lqcd.STAGGERED and not args.no_variants and solver_variants:
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
        # The time-slab decomposition with all R slabs on THIS GPU, driven in
        # lock-step on one stream: the kernels, peer stores and mailboxes of an R-GPU run, so the
        # difference to the undivided solve is the cost of the decomposition itself (6 tiny kernels
        # per iteration, smaller grids), not of any link.  One warm-up + one timed solve each.
        if world == 1 and not mixed and full:
            from paper_1311_2719_b200 import slab as slab_mod
            ug, bg = torch.from_numpy(u), torch.from_numpy(b)
            for R in (2, 4, 8):
                if cfg["dims"][3] % R or (cfg["dims"][3] // R) % 2 or cfg["dims"][3] // R < 2:
                    continue
                try:   # an extra, never allowed to take the headline line down with it
                    variants["slab_group%d_on_one_gpu" % R] = slab_group_variant(slab_mod, cfg, ug, bg, R, args, maxiter)
                except Exception as exc:  # noqa: BLE001
                    variants["slab_group%d_on_one_gpu" % R] = {"error": repr(exc)[:200]}
            try:   # the mixed-precision slab solver (separate launches per synchronisation point), two slabs
                variants["slab_group2_mixed_on_one_gpu"] = slab_group_variant(slab_mod, cfg, ug, bg, 2, args, maxiter, mixed=True)
            except Exception as exc:  # noqa: BLE001
                variants["slab_group2_mixed_on_one_gpu"] = {"error": repr(exc)[:200]}

    if f == lqcd.WILSON and not args.no_variants and solver_variants:
        # the even-odd (Schur) preconditioned solver of the same system M x = b, and two-row links
        variants = {}
        for recon_v in (args.recon, 30 - args.recon):
            lat.set_option(lqcd.OPT_RECONSTRUCT, recon_v)
            lat.load_gauge(u_dev)
            for name_v, call_v in (("eo_solve", lambda: lat.wilson_solve_eo(cfg["param"], cfg["tol"], maxiter, b_dev)),
                                   ("f64", lambda: lat.cg_solve(cfg["param"], cfg["tol"], maxiter, b_dev, x_dev))):
                if name_v == "f64" and recon_v == args.recon:
                    continue   # the headline itself
                call_v()
                v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                barrier()
                v0.record(lat.stream)
                _, it_v, res_v, st_v = call_v()
                v1.record(lat.stream)
                barrier()
                variants["%s_recon%d" % (name_v, recon_v)] = {"time_to_solution_ms": max_over_ranks(v0.elapsed_time(v1)), "iters": it_v,
                                                              "true_residual": res_v, "converged": st_v == 0}
        lat.set_option(lqcd.OPT_RECONSTRUCT, args.recon)
        lat.load_gauge(u_dev)

    # ---- the oracle beside it (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and full:
        r = oracle_arm(cfg, u, b, steps=2, warmup=0, target_seconds=6.0)
        cpu = {"value": r["value"], "unit": "GB/s", "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
               "dslash": oracle_dslash_times(cfg, u, b)}   # per call, all cores and one thread, beside dslash.us_per_call

    if cpu is None and not full and rank == 0 and world == 1 and not args.no_cpu_baseline and cfg["name"] in ("cfg1", "cfg2", "cfg3"):
        # --all-configs: the oracle's hopping term per call (all cores, one thread) for configs 1-3, SURVEY 8(d)
        cpu = {"value": None, "unit": "GB/s", "kind": "oracle", "sample": "hopping term only",
               "dslash": oracle_dslash_times(cfg, u, b, budget_s=2.0)}
        cpu["cores"] = cpu["dslash"]["cores"]
    line = {
        "metric": metric, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_solve, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64" if not mixed else "f32 iterations + f64 reliable updates",
        "data": "synthetic",
        "config": config_dict(args, cfg, world),
        "cg": {"time_to_solution_ms": ms_solve, "iters": iters, "reliable_updates": updates if mixed else None,
               "true_residual": res, "path": path_ran,   # lqcd_last_cg_path(): the loop that really ran
               "us_per_iteration": ms_solve * 1e3 / max(iters, 1)},
        "dslash": {"us_per_call": us_dslash, "GBps": achieved, "GFLOPs": dflops * sites_out / (us_dslash * 1e-6) / 1e9,
                   "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS, "reps": args.dslash_reps},
        "roofline": {"bound": "hbm", "kernel": "stag_dslash_kernel<SE_PLAIN>" if f == lqcd.STAGGERED else
                     "wilson_dslash_kernel<WE_PLAIN>", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "peak_source": peak_src, "traffic": None, "traffic_source": None,
                     "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                     "note": "peak = a copy (half its bytes are writes); this kernel is 96 % reads and its 48 B/site input is the "
                             "previous launch's output (L2-resident in the ping-pong sweep), so frac can exceed 1: "
                             "without that input 1200/1248 of it, on ncu DRAM bytes traffic/time",
                     "bytes_per_site": dbytes, "sites_per_launch": sites_out},
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "cpu_baseline": cpu, "variants": variants,
    }
    if path_ran != line["config"]["cg_path"]:   # the library chose otherwise than bench.py's copy of its rule: say so
        line["config"]["cg_path"] = path_ran
        line["config"]["cg_mode"] = "%s (lqcd_last_cg_path: %s)" % (args.cg_mode, path_ran)
    line["roofline"]["traffic"] = ncu_traffic("%s_dslash_plain%s" % (cfg["name"], "" if args.recon == 18 else "_recon12"))
    if line["roofline"]["traffic"] is not None:
        line["roofline"]["traffic_source"] = "profiles/traffic.csv (ncu --set full, builder-run; not measured by this run)"
    if world > 1 and full and f == lqcd.STAGGERED and not mixed:
        # N > 1: replicas stay the headline (BASELINE.json: everything runs on one GPU); beside it ONE solve of the same
        # system cut into N time-slabs through lqcd_slab_cg_solve (IPC-mapped mailboxes, halo stores and sums through
        # peer memory: what replaces the paper's host-staged MPI_ALLGATHER).  First run on real
        # peers: bounded waits (LQCD_ECOMM) and try/except keep a failure out of the headline line.
        sv = slab_strong_variant(args, cfg, ranks, device, maxiter)
        if rank == 0:
            line["variants"] = dict(line["variants"] or {}, **{"slab_strong_x%d" % world: sv})
    lat.close()
    return line


def config_entry(line):
    """What the default line's `configs` object keeps of one config's full line (same code, same timing rules)."""
    e2e, ck = line.get("e2e") or {}, line.get("clocks") or {}
    out = {"workload": line["config"]["workload"], "cg_path": line["cg"]["path"], "l2_policy": line["config"]["l2_policy"],
           "steps": line["steps"], "warmup": line["warmup"],
           "cg_ms": line["ms_per_step"], "iters": line["cg"]["iters"], "true_residual": line["cg"]["true_residual"],
           "us_per_iteration": line["cg"]["us_per_iteration"], "value_GBps": line["value"],
           "dslash_us": line["dslash"]["us_per_call"], "dslash_GBps": line["dslash"]["GBps"],
           "dslash_GFLOPs": line["dslash"]["GFLOPs"], "dslash_frac_of_peak": line["roofline"]["frac"],
           "dslash_kernel": line["roofline"]["kernel"], "e2e_ms": e2e.get("ms_per_step"),
           "gpu_launches": line["gpu_launches"], "clocks": ck}
    if line.get("variants"):
        out["variants"] = {k: {"time_to_solution_ms": v.get("time_to_solution_ms"), "iters": v.get("iters"),
                               "reliable_updates": v.get("reliable_updates"), "true_residual": v.get("true_residual"),
                               "converged": v.get("converged")} for k, v in line["variants"].items()}
    return out


def all_configs_table(lines):
    """Markdown table of an --all-configs run (one row per BASELINE.json config)."""
    out = ["| config | CG time to solution | iterations | true residual | us per iteration | `value` GB/s | plain Dslash us "
           "(GB/s, of measured copy peak) | oracle Dslash us per call: all cores / one thread | e2e (host buffers) | "
           "SM clock MHz (reasons) |", "|---|---|---|---|---|---|---|---|---|---|"]
    for l in lines:
        e2e = "%.2f ms" % l["e2e"]["ms_per_step"] if l.get("e2e") else "--"
        ck = l.get("clocks") or {}
        od = (l.get("cpu_baseline") or {}).get("dslash")
        ods = "%.0f (%d cores) / %.0f" % (od["us_per_call_all_cores"], od["cores"], od["us_per_call_one_thread"]) if od else "--"
        out.append("| %s | %.3f ms | %d | %.2e | %.2f | %.0f | %.2f (%.0f, %.3f) | %s | %s | %s (%s) |" % (
            l["config"]["workload"], l["ms_per_step"], l["cg"]["iters"], l["cg"]["true_residual"], l["cg"]["us_per_iteration"],
            l["value"], l["dslash"]["us_per_call"], l["dslash"]["GBps"], l["roofline"]["frac"], ods, e2e,
            ck.get("sm_mhz"), ",".join(ck.get("reasons") or []) or "none"))
    return "\n".join(out) + "\n"


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
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: replicas = independent right-hand sides per GPU (weak scaling, the default); "
                         "slab = ONE system cut into time-slabs, halo exchange and sums through peer memory "
                         "(strong scaling; include/lqcd_slab.h; staggered configs)")
    ap.add_argument("--all-configs", action="store_true",
                    help="the five BASELINE.json configs in one run (no variants, no oracle timing): one JSON line with a list")
    ap.add_argument("--table", default=None, help="with --all-configs: also write the five-config table (markdown) to this file")
    ap.add_argument("--no-configs", action="store_true",
                    help="N = 1 default line: skip the `configs` object (the other four BASELINE.json configs timed by the same code)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    cfg = synth.config(args.config)
    workload = workload_name(cfg)
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
                "config": config_dict(args, cfg, 1),
                "cpu_baseline": {"value": r["value"], "unit": "GB/s", "cores": r["cores"], "kind": "oracle",
                                 "sample": r["sample"], "dslash": oracle_dslash_times(cfg, u, b)},
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

    if args.parallelism == "slab":
        return slab_arm(args, cfg, workload, metric, ranks, device)

    if args.all_configs:
        # one process, the five BASELINE.json configs one after the other (no variants, no oracle timing):
        # the table of profiles/ is written from this one line
        lines = [ours_line(args, synth.config(n), metric, ranks, device, lqcd, torch, full=False) for n in (1, 2, 3, 4, 5)]
        if rank == 0:
            print(json.dumps({"metric": metric, "unit": "GB/s", "n_gpus": world, "all_configs": lines}))
            if args.table:
                with open(args.table, "w") as fh:
                    fh.write(all_configs_table(lines))
        ranks.close()
        return 0
    line = ours_line(args, cfg, metric, ranks, device, lqcd, torch, full=True)
    if world == 1 and not args.no_configs and args.config == 3 and args.precision == "f64" and args.recon == 18:
        # north_star: throughput "on all five configs".  The headline (value, roofline, e2e) stays config 3; the other
        # four are timed here by the same code and rules (>= 3 warm-up solves, args.steps timed solves, device events,
        # own clock record), each reduced to a few numbers; configs 4 and 5 with their other solvers (even-odd Wilson;
        # two-row links and mixed precision).  A failure here never takes the headline down.
        line["configs"] = {}
        for n in (1, 2, 4, 5):
            c = synth.config(n)
            t0 = time.perf_counter()
            try:
                entry = config_entry(ours_line(args, c, metric, ranks, device, lqcd, torch, full=False, solver_variants=n in (4, 5)))
            except Exception as exc:  # noqa: BLE001
                entry = {"error": repr(exc)[:300]}
            entry["wall_s_including_input_generation"] = time.perf_counter() - t0
            line["configs"][c["name"]] = entry
            torch.cuda.empty_cache()
    if rank == 0:
        print(json.dumps(line))
    ranks.close()
    return 0


if __name__ == "__main__":
    sys.exit(main())
