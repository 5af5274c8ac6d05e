"""Test-side lattice helpers written independently of oracle/ and of the CUDA library:
vectorised numpy statements of the site ordering of SURVEY.md 8(b), used to pin the
oracle's tables and to build plane waves / gauge transformations."""
import numpy as np


def site_coordinates(dims):
    """x[g][mu] for the canonical index g = parity*Vh + s//2, s lexicographic with x0 fastest."""
    L0, L1, L2, L3 = dims
    v = L0 * L1 * L2 * L3
    s = np.arange(v, dtype=np.int64)
    x = np.stack([s % L0, (s // L0) % L1, (s // (L0 * L1)) % L2, s // (L0 * L1 * L2)], axis=1)
    g = (x.sum(axis=1) % 2) * (v // 2) + s // 2
    out = np.empty((v, 4), np.int64)
    out[g] = x
    return out


def site_index(dims, x):
    """canonical g of integer coordinates x[...,4] (already wrapped into range)."""
    L0, L1, L2, L3 = dims
    v = L0 * L1 * L2 * L3
    s = x[..., 0] + L0 * (x[..., 1] + L1 * (x[..., 2] + L2 * x[..., 3]))
    return (x.sum(axis=-1) % 2) * (v // 2) + s // 2


def shifted_index(dims, mu, sign):
    """g-index of x + sign*mu_hat for every g (periodic)."""
    x = site_coordinates(dims).copy()
    x[:, mu] = (x[:, mu] + sign) % dims[mu]
    return site_index(dims, x)


def momenta(dims, n):
    """p_mu = 2 pi n_mu / L_mu for mu<3 and 2 pi (n_3 + 1/2) / L_3 (antiperiodic time)."""
    n = np.asarray(n, dtype=np.float64)
    L = np.asarray(dims, dtype=np.float64)
    p = 2.0 * np.pi * n / L
    p[3] = 2.0 * np.pi * (n[3] + 0.5) / L[3]
    return p


def read_gammas(path):
    val = {"0": 0, "1": 1, "-1": -1, "i": 1j, "-i": -1j}
    gam = np.zeros((4, 4, 4), complex)
    mu, row = -1, 0
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("gamma"):
            mu, row = int(line.split()[1]), 0
            continue
        gam[mu, row] = [val[t] for t in line.split()]
        row += 1
    return gam


# ------------------------------------------------------------------ stored oracle references
import json as _json
import os as _os

GOLDEN = _os.path.join(_os.path.dirname(_os.path.abspath(__file__)), "golden", "oracle_cg_reference.json")


def golden(key):
    """Entry `key` ("cfg3", "cfg5", "cfg3_mixed", ...) of tests/golden/oracle_cg_reference.json (written by
    tests/golden/make_golden.py from oracle/ alone).  A missing file or entry FAILS the test: parity against
    the oracle's CG is part of the contract on every BASELINE.json config."""
    assert _os.path.exists(GOLDEN), "tests/golden/oracle_cg_reference.json is missing: run tests/golden/make_golden.py"
    ref = _json.load(open(GOLDEN))
    assert key in ref, "no stored oracle reference for %s: run tests/golden/make_golden.py" % key
    return ref[key]


def check_sampled_solution(x, ref, tol):
    """The stored sample of the oracle's solution (>= 4096 entries on the full-size configs) against the
    same entries of `x`: |x_S - want_S| <= tol |x_oracle| sqrt(|S| / n), the sampled form of rel-L2 <= tol
    (no slack factor), and the norm of the whole vector."""
    import numpy as np
    idx = np.asarray(ref["sample_index"])
    want = np.asarray(ref["sample_re"]) + 1j * np.asarray(ref["sample_im"])
    got = x.ravel()[idx]
    assert np.linalg.norm(got - want) <= tol * ref["x_norm"] * np.sqrt(len(idx) / x.size)
    assert abs(np.linalg.norm(x.ravel()) - ref["x_norm"]) <= tol * ref["x_norm"]
