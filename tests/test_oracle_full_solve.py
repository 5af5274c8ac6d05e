"""Pins for the oracle's full-system staggered solve M x = b, M = m + D.

P10: the even-odd reduction (source preparation, CG on the even sites, reconstruction of the odd
sites) must give the solution of the *un-reduced* system.  The un-reduced system is built here from
the bare hopping term (pinned by P1-P4) plus m on the diagonal, and solved by Gaussian elimination
(numpy) or checked by its residual -- never through the reduction formulas under test.  No GPU needed.
"""
import numpy as np
import pytest

import oracle
from oracle import STAGGERED
from paper_1311_2719_b200 import synth


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def dense_full_M(dims, u, mass):
    """(2n x 2n) matrix of m + D in the basis (even block, odd block), column by column from oracle.dslash."""
    vh = synth.volume(dims) // 2
    n = 3 * vh
    m = np.zeros((2 * n, 2 * n), complex)
    for j in range(n):
        e = np.zeros((3, vh), complex)
        e.ravel()[j] = 1.0
        m[n:, j] = oracle.dslash(dims, STAGGERED, u, 1, e).ravel()   # D_oe acting on an even unit vector
        m[:n, n + j] = oracle.dslash(dims, STAGGERED, u, 0, e).ravel()  # D_eo acting on an odd unit vector
    m += mass * np.eye(2 * n)
    return m


def full_source(dims, seed):
    return synth.source(dims, "staggered", seed), synth.source(dims, "staggered", seed + 1)


@pytest.mark.parametrize("dims,kind,mass", [((2, 2, 2, 2), "haar", 0.1), ((2, 2, 2, 2), "smooth", 0.05),
                                            ((4, 2, 2, 2), "random_su3", 0.3)])
def test_full_solve_against_dense_elimination(dims, kind, mass):
    u = synth.gauge_field(dims, kind, 71)
    be, bo = full_source(dims, 72)
    m = dense_full_M(dims, u, mass)
    # D is anti-hermitian, so M^+ = m - D (the statement the reduction rests on)
    assert np.allclose(m + m.conj().T, 2 * mass * np.eye(m.shape[0]), atol=1e-14)
    x = np.linalg.solve(m, np.concatenate([be.ravel(), bo.ravel()]))
    r = oracle.stag_solve_full(dims, u, mass, 1e-13, 2000, be, bo)
    assert r["status"] == 0
    n = be.size
    assert rel(r["x_e"].ravel(), x[:n]) < 1e-10
    assert rel(r["x_o"].ravel(), x[n:]) < 1e-10
    assert r["true_residual"] < 1e-11


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_full_solve_residual_from_bare_hopping_term(dims):
    mass = 0.1
    u = synth.gauge_field(dims, "haar", 73)
    be, bo = full_source(dims, 74)
    r = oracle.stag_solve_full(dims, u, mass, 1e-10, 5000, be, bo)
    assert r["status"] == 0
    # M x from the bare hopping term, not from oracle.stag_M
    me = mass * r["x_e"] + oracle.dslash(dims, STAGGERED, u, 0, r["x_o"])
    mo = mass * r["x_o"] + oracle.dslash(dims, STAGGERED, u, 1, r["x_e"])
    res = np.sqrt((np.linalg.norm(be - me) ** 2 + np.linalg.norm(bo - mo) ** 2) /
                  (np.linalg.norm(be) ** 2 + np.linalg.norm(bo) ** 2))
    assert res < 2e-9      # |r'|/(m |b|) with |r'| <= 1e-10 |b'|, |b'| <~ |b| (m + |D|)
    assert abs(res - r["true_residual"]) <= 1e-3 * res + 1e-16
    # stag_M itself against the same construction
    ge, go = oracle.stag_M(dims, u, mass, r["x_e"], r["x_o"])
    assert rel(ge, me) < 1e-15 and rel(go, mo) < 1e-15
    # the even half solves the reduced system A x_e = m b_e - D_eo b_o
    bp = mass * be - oracle.dslash(dims, STAGGERED, u, 0, bo)
    assert rel(oracle.apply_MdagM(dims, STAGGERED, u, mass, r["x_e"]), bp) < 1e-9


def test_full_solve_free_field_plane_wave():
    """U = 1: on a plane wave M^+M = m^2 + sum sin^2 p, so x = M^+ b / (m^2 + sum sin^2 p) in closed form."""
    import lattice_util as lu
    dims, mass = (4, 4, 2, 4), 0.2
    v = synth.volume(dims)
    vh = v // 2
    u = np.broadcast_to(np.eye(3, dtype=complex), (v, 4, 3, 3)).copy()
    x = lu.site_coordinates(dims)
    p = lu.momenta(dims, (1, 3, 0, 2))
    c = np.array([0.3 - 1j, 2.0, -0.5j])
    wave = np.exp(1j * (x @ p))
    b = c[:, None] * wave[None, :]
    be, bo = np.ascontiguousarray(b[:, :vh]), np.ascontiguousarray(b[:, vh:])
    lam = mass ** 2 + np.sum(np.sin(p) ** 2)
    # M^+ b = m b - D b from the bare hopping term
    mdb_e = mass * be - oracle.dslash(dims, STAGGERED, u, 0, bo)
    mdb_o = mass * bo - oracle.dslash(dims, STAGGERED, u, 1, be)
    r = oracle.stag_solve_full(dims, u, mass, 1e-13, 500, be, bo)
    assert rel(r["x_e"], mdb_e / lam) < 1e-11 and rel(r["x_o"], mdb_o / lam) < 1e-11


def test_full_solve_edge_cases():
    dims = (2, 2, 2, 2)
    u = synth.gauge_field(dims, "haar", 75)
    z = np.zeros((3, 8), complex)
    r = oracle.stag_solve_full(dims, u, 0.1, 1e-10, 10, z, z)
    assert r["status"] == 0 and r["iters"] == 0 and r["true_residual"] == 0
    assert not r["x_e"].any() and not r["x_o"].any()
    be, bo = full_source(dims, 76)
    with pytest.raises(ValueError):
        oracle.stag_solve_full(dims, u, 0.0, 1e-10, 10, be, bo)
    # source on the odd sites only: the even source of the reduced system is -D_eo b_o
    r = oracle.stag_solve_full(dims, u, 0.1, 1e-12, 500, z, bo)
    me, mo = oracle.stag_M(dims, u, 0.1, r["x_e"], r["x_o"])
    assert np.linalg.norm(me) < 1e-10 * np.linalg.norm(bo) and rel(mo, bo) < 1e-10
