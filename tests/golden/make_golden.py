#!/usr/bin/env python
"""Write tests/golden/oracle_cg_reference.json: what the CPU ORACLE's conjugate gradient gives on
the BASELINE.json configs (iteration count, true residual, norm of the solution and a few
sampled solution entries).  Calls only oracle/ and the seeded input generators; nothing here
touches the CUDA library.  Usage: python tests/golden/make_golden.py [cfg ...]   (default 1 2 3 4)
       python tests/golden/make_golden.py --mixed [cfg ...]   adds "cfgN_mixed": the oracle's
       mixed-precision CG (delta = 0.1) on the staggered configs: iterations, reliable updates, residual.

The full-size GPU tests compare against these instead of re-running minutes of oracle CG.
LAPACK rounding in the input generators may differ in the last bit between machines; the CG
tolerances (solution 1e-9, iterations +-2) absorb that.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1311_2719_b200 import synth  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_cg_reference.json")


def dump(ref):
    """One key per line, number lists on one line (the 4096-entry samples stay readable in a diff)."""
    lines = []
    for name in sorted(ref):
        items = ",\n".join('  %s: %s' % (json.dumps(k), json.dumps(ref[name][k])) for k in sorted(ref[name]))
        lines.append(' %s: {\n%s\n }' % (json.dumps(name), items))
    with open(OUT, "w") as f:
        f.write("{\n" + ",\n".join(lines) + "\n}\n")
NSAMPLE = 4096     # cfg 1, 2, 4 (re-run in full inside the GPU tests) were written with 64


def mixed(cfgs):
    ref = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for n in cfgs:
        c, u, b = synth.config_inputs(n)
        assert c["fermion"] == "staggered"
        t0 = time.time()
        r = oracle.cg_mixed(c["dims"], u, c["param"], c["tol"], 100000, b, delta=0.1)
        dt = time.time() - t0
        x = r["x"].ravel()
        ref["cfg%d_mixed" % n] = {
            "delta": 0.1, "iters": r["iters"], "updates": r["updates"], "status": r["status"],
            "true_residual": r["true_residual"], "x_norm": float(np.linalg.norm(x)), "oracle_seconds": round(dt, 1),
        }
        print("cfg%d mixed: iters %d, updates %d, true residual %.3e, %.1f s"
              % (n, r["iters"], r["updates"], r["true_residual"], dt), flush=True)
        dump(ref)


def main():
    if "--mixed" in sys.argv:
        return mixed([int(a) for a in sys.argv[1:] if a != "--mixed"] or [1, 2, 3])
    cfgs = [int(a) for a in sys.argv[1:]] or [1, 2, 3, 4]
    ref = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for n in cfgs:
        c, u, b = synth.config_inputs(n)
        f = 0 if c["fermion"] == "staggered" else 1
        t0 = time.time()
        r = oracle.cg(c["dims"], f, u, c["param"], c["tol"], 100000, b)
        dt = time.time() - t0
        x = r["x"].ravel()
        idx = np.random.default_rng(1311 + n).choice(x.size, min(NSAMPLE, x.size), replace=False)
        idx.sort()
        ref["cfg%d" % n] = {
            "dims": list(c["dims"]), "fermion": c["fermion"], "links": c["links"], "param": c["param"],
            "tol": c["tol"], "seed": c["seed"], "iters": r["iters"], "status": r["status"],
            "true_residual": r["true_residual"], "x_norm": float(np.linalg.norm(x)),
            "sample_index": [int(i) for i in idx], "sample_re": [float(v) for v in x[idx].real],
            "sample_im": [float(v) for v in x[idx].imag], "oracle_seconds": round(dt, 1),
            "oracle_threads": oracle.num_threads(),
        }
        print("cfg%d: iters %d, true residual %.3e, %.1f s" % (n, r["iters"], r["true_residual"], dt), flush=True)
        dump(ref)


if __name__ == "__main__":
    main()
