"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no Dslash, no CG, no lattice
geometry): it only draws SU(3) link matrices and Gaussian sources as flat arrays
indexed by the canonical site index g; what g means
geometrically is the business of the oracle and of the CUDA library, each on its
own.  The gauge ensembles of arXiv 1311.2719 are unpublished (§6 gives
neither lattice sizes nor couplings), so these fields stand in for them, with the
recipes BASELINE.json `configs` states in words:

* ``random_su3`` (cfg 1): Z 3x3 with Re,Im ~ N(0,1); Gram-Schmidt the rows in
  order; divide the third row by the determinant.
* ``smooth`` (cfg 2,4,5): G = Z/sqrt(2); H = (G+G^+)/2 - tr/3; U = exp(i*eps*H).
* ``haar`` (cfg 3): Z = QR; Q <- Q diag(r_ii/|r_ii|); last column /= det(Q).
* sources: Re,Im ~ N(0,1) per component.

Draws are made chunk by chunk over g (CHUNK sites per chunk, one child generator
per chunk from ``SeedSequence(seed).spawn``) so that the result does not depend
on how many threads build it.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

CHUNK = 16384  # sites per independently seeded chunk

SEED_BASE = 13112719 * 10

# BASELINE.json `configs`, 1-based like the survey's "cfg" numbers.
CONFIGS = {
    1: dict(dims=(4, 4, 4, 4), fermion="staggered", links="random_su3", param=0.1, tol=1e-10),
    2: dict(dims=(16, 16, 16, 16), fermion="staggered", links="smooth", param=0.05, tol=1e-10),
    3: dict(dims=(32, 32, 32, 32), fermion="staggered", links="haar", param=0.01, tol=1e-10),
    4: dict(dims=(16, 16, 16, 32), fermion="wilson", links="smooth", param=0.12, tol=1e-10),
    5: dict(dims=(48, 48, 48, 96), fermion="staggered", links="smooth", param=0.005, tol=1e-10),
}


def config(n: int) -> dict:
    """Parameters of BASELINE.json config n (1..5) plus its seed."""
    c = dict(CONFIGS[n])
    c["seed"] = SEED_BASE + n
    c["name"] = "cfg%d" % n
    return c


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def _normal_complex(rng, shape):
    z = rng.standard_normal(tuple(shape) + (2,))
    return z.view(np.complex128)[..., 0]


def _dagger(a):
    return np.conj(np.swapaxes(a, -1, -2))


def _det3(a):
    return (a[..., 0, 0] * (a[..., 1, 1] * a[..., 2, 2] - a[..., 1, 2] * a[..., 2, 1])
            - a[..., 0, 1] * (a[..., 1, 0] * a[..., 2, 2] - a[..., 1, 2] * a[..., 2, 0])
            + a[..., 0, 2] * (a[..., 1, 0] * a[..., 2, 1] - a[..., 1, 1] * a[..., 2, 0]))


def _gram_schmidt_rows(z):
    r0 = z[:, 0, :]
    r0 = r0 / np.linalg.norm(r0, axis=1, keepdims=True)
    r1 = z[:, 1, :]
    r1 = r1 - np.sum(np.conj(r0) * r1, axis=1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=1, keepdims=True)
    r2 = z[:, 2, :]
    r2 = r2 - np.sum(np.conj(r0) * r2, axis=1, keepdims=True) * r0
    r2 = r2 - np.sum(np.conj(r1) * r2, axis=1, keepdims=True) * r1
    r2 = r2 / np.linalg.norm(r2, axis=1, keepdims=True)
    return np.stack([r0, r1, r2], axis=1)


def _links_random_su3(rng, n):
    z = _normal_complex(rng, (n, 3, 3))
    u = _gram_schmidt_rows(_gram_schmidt_rows(z))  # second pass only removes rounding
    u[:, 2, :] /= _det3(u)[:, None]
    return u


def _links_smooth(rng, n, eps):
    g = _normal_complex(rng, (n, 3, 3)) / np.sqrt(2.0)
    h = 0.5 * (g + _dagger(g))
    tr = (h[:, 0, 0] + h[:, 1, 1] + h[:, 2, 2]) / 3.0
    for i in range(3):
        h[:, i, i] -= tr
    w, v = np.linalg.eigh(h)
    return (v * np.exp(1j * eps * w)[:, None, :]) @ _dagger(v)


def _links_haar(rng, n):
    z = _normal_complex(rng, (n, 3, 3))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=1, axis2=2)
    q = q * (d / np.abs(d))[:, None, :]
    q[:, :, 2] /= _det3(q)[:, None]
    return q


def gauge_field(dims, kind: str, seed: int, eps: float = 0.3, threads: int | None = None) -> np.ndarray:
    """Links in the canonical layout u[g][mu][row][col], complex128, shape (V,4,3,3)."""
    v = volume(dims)
    out = np.empty((v, 4, 3, 3), dtype=np.complex128)
    if kind == "unit":
        out[...] = np.eye(3)
        return out
    nchunk = (v + CHUNK - 1) // CHUNK
    children = np.random.SeedSequence(seed).spawn(nchunk)

    def work(i):
        lo = i * CHUNK
        hi = min(v, lo + CHUNK)
        rng = np.random.default_rng(children[i])
        n = (hi - lo) * 4
        if kind == "random_su3":
            u = _links_random_su3(rng, n)
        elif kind == "smooth":
            u = _links_smooth(rng, n, eps)
        elif kind == "haar":
            u = _links_haar(rng, n)
        else:
            raise ValueError("unknown link ensemble %r" % (kind,))
        out[lo:hi] = u.reshape(hi - lo, 4, 3, 3)

    nthr = threads or min(nchunk, os.cpu_count() or 1)
    if nthr <= 1 or nchunk == 1:
        for i in range(nchunk):
            work(i)
    else:
        with ThreadPoolExecutor(nthr) as ex:
            list(ex.map(work, range(nchunk)))
    return out


def source(dims, fermion: str, seed: int) -> np.ndarray:
    """Gaussian source: staggered -> (3, Vh) on the even sites; wilson -> (4, 3, V)."""
    v = volume(dims)
    rng = np.random.default_rng(np.random.SeedSequence([seed, 0x50CE]))
    if fermion == "staggered":
        return _normal_complex(rng, (3, v // 2))
    if fermion == "wilson":
        return _normal_complex(rng, (4, 3, v))
    raise ValueError("unknown fermion type %r" % (fermion,))


def vector(shape, seed: int) -> np.ndarray:
    """Any other Gaussian complex test vector."""
    rng = np.random.default_rng(np.random.SeedSequence([seed, 0xFEC7]))
    return _normal_complex(rng, shape)


def su3_field(n: int, seed: int) -> np.ndarray:
    """n Haar SU(3) matrices, shape (n,3,3): the g(x) of a gauge transformation."""
    rng = np.random.default_rng(np.random.SeedSequence([seed, 0x6A06]))
    return _links_haar(rng, n)


def config_inputs(n: int, threads: int | None = None):
    """(cfg dict, gauge field, source) of BASELINE.json config n."""
    c = config(n)
    u = gauge_field(c["dims"], c["links"], c["seed"], threads=threads)
    b = source(c["dims"], c["fermion"], c["seed"])
    return c, u, b
