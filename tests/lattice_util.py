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
