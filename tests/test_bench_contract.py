"""bench.py's contract that can be checked without a GPU: the reference arm (the oracle on the host
cores) prints one JSON line with the agreed keys, and the byte model behind `value` is the one
DESIGN.md / SURVEY.md 8(d) state."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_byte_model_matches_the_survey_figures():
    import bench
    from paper_1311_2719_b200 import synth
    c3, c4 = synth.config(3), synth.config(4)
    vh = synth.volume(c3["dims"]) // 2
    # per iteration and site: 2 x 1152 B of links + 11 vector passes x 48 B = 2832 B (two-row links: 2064 B)
    assert bench.cg_bytes(c3, 11) - bench.cg_bytes(c3, 10) == 2832 * vh
    assert bench.cg_bytes(c3, 11, recon=12) - bench.cg_bytes(c3, 10, recon=12) == 2064 * vh
    # fp32 iterations of the mixed solver: half of that
    assert bench.cg_bytes(c3, 11, 18, updates=2) - bench.cg_bytes(c3, 10, 18, updates=2) == 1416 * vh
    assert bench.cg_bytes(c3, 11, 12, updates=2) - bench.cg_bytes(c3, 10, 12, updates=2) == 1032 * vh
    # Wilson: two full-lattice hops + 11 passes over 192 B spinors
    v = synth.volume(c4["dims"])
    assert bench.cg_bytes(c4, 6) - bench.cg_bytes(c4, 5) == (2 * 1152 + 11 * 192) * v
    assert bench.STAG_DSLASH_BYTES == 8 * 144 + 48 + 48 and bench.WILSON_DSLASH_BYTES == 8 * 144 + 192 + 192
    assert bench.STAG_DSLASH_FLOPS == 8 * 66 + 7 * 6 and bench.WILSON_DSLASH_FLOPS == 8 * (12 + 2 * 66) + 7 * 24


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"):
        assert key in line, key
    assert line["impl"] == "reference" and line["unit"] == "GB/s" and line["value"] > 0 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
    assert "workload" in line["config"] and "cfg1" in line["config"]["workload"]
    # both arms carry the same config keys (what the reference arm samples is said in cpu_baseline.sample)
    import argparse
    import bench
    from paper_1311_2719_b200 import synth
    ours = bench.config_dict(argparse.Namespace(precision="f64", recon=18, cg_mode="graph", check_every=8), synth.config(1), 1)
    assert line["config"] == ours
    # the oracle's hopping term alone, per call, on all cores and on one thread (SURVEY 8(d) timing protocol)
    d = line["cpu_baseline"]["dslash"]
    assert d["us_per_call_all_cores"] > 0 and d["us_per_call_one_thread"] > 0 and d["cores"] == line["cpu_baseline"]["cores"]


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--gpus", "2"],
                         capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_config_says_which_loop_runs_and_whether_the_workload_is_l2_resident():
    """bench.py's copy of the library's rule (one cooperative kernel where the stored links take at most a third of the
    L2; never against an explicit --cg-mode sync; fp64 staggered solves only) and the l2_policy derived from the link
    bytes.  The GPU arm checks the rule against lqcd_last_cg_path() and overrides `config` if the library chose otherwise."""
    import argparse
    import bench
    from paper_1311_2719_b200 import synth
    ns = lambda **kw: argparse.Namespace(**dict(dict(precision="f64", recon=18, cg_mode="graph", check_every=8), **kw))
    want = {1: "persistent", 2: "persistent", 3: "host_loop", 4: "host_loop", 5: "host_loop"}
    for n, path in want.items():
        c = bench.config_dict(ns(), synth.config(n), 1)
        assert c["cg_path"] == path and (c["check_every"] is None) == (path == "persistent")
        assert ("L2-RESIDENT" in c["l2_policy"]) == (path == "persistent")
        assert ("larger than L2" in c["l2_policy"]) == (n in (3, 5))
    assert bench.config_dict(ns(cg_mode="sync"), synth.config(2), 1)["cg_path"] == "host_loop"
    assert bench.config_dict(ns(precision="mixed"), synth.config(2), 1)["cg_path"] == "host_loop"
    # what `configs` keeps of a full line
    line = {"config": {"workload": "w", "l2_policy": "p"}, "cg": {"path": "host_loop", "iters": 5, "true_residual": 1e-11,
            "us_per_iteration": 2.0}, "steps": 3, "warmup": 3, "ms_per_step": 0.01, "value": 1.0,
            "dslash": {"us_per_call": 1.0, "GBps": 2.0, "GFLOPs": 3.0}, "roofline": {"frac": 0.5, "kernel": "k"},
            "e2e": {"ms_per_step": 0.02}, "gpu_launches": 7, "clocks": {"sm_mhz": 1965.0},
            "variants": {"v": {"time_to_solution_ms": 1.0, "iters": 5, "GBps": 9.0}}}
    e = bench.config_entry(line)
    assert e["cg_ms"] == 0.01 and e["iters"] == 5 and e["dslash_frac_of_peak"] == 0.5 and e["e2e_ms"] == 0.02
    assert e["variants"]["v"]["time_to_solution_ms"] == 1.0 and e["cg_path"] == "host_loop"
