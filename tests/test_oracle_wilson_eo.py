"""Pins for the oracle's even-odd (Schur) preconditioned Wilson solve of M x = b.

P12: the Schur complement and the reduction must reproduce the *un-reduced* system, which is built here
from the full-lattice M = 1 - kappa D_W (pinned by P4-P7) and solved by Gaussian elimination, or checked
by its residual; the free-field closed form pins the operator itself.  No GPU needed.
"""
import numpy as np
import pytest

import oracle
from oracle import WILSON
from paper_1311_2719_b200 import synth

import lattice_util as lu


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def even_only(v, vh):
    out = v.copy()
    out[:, :, vh:] = 0
    return out


@pytest.mark.parametrize("dims,kind,kappa", [((2, 2, 2, 2), "smooth", 0.12), ((2, 2, 2, 2), "haar", 0.1),
                                             ((2, 2, 2, 4), "random_su3", 0.11)])
def test_eo_solve_against_dense_elimination_of_the_full_matrix(dims, kind, kappa):
    u = synth.gauge_field(dims, kind, 121)
    b = synth.source(dims, "wilson", 122)
    n = b.size
    m = np.empty((n, n), complex)
    for j in range(n):
        e = np.zeros(n, complex)
        e[j] = 1.0
        m[:, j] = oracle.wilson_M(dims, u, kappa, e.reshape(b.shape)).ravel()
    x_dense = np.linalg.solve(m, b.ravel()).reshape(b.shape)
    r = oracle.wilson_solve_eo(dims, u, kappa, 1e-13, 5000, b)
    assert r["status"] == 0
    assert rel(r["x"], x_dense) < 1e-10
    assert r["true_residual"] < 1e-11


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4)])
def test_schur_identity_and_adjoint(dims):
    kappa = 0.12
    v = synth.volume(dims)
    vh = v // 2
    u = synth.gauge_field(dims, "haar", 123)
    xe = even_only(synth.source(dims, "wilson", 124), vh)
    # M applied to (x_e, x_o = kappa D_oe x_e) gives (Mhat x_e, 0): the defining property of the Schur complement
    full = xe.copy()
    full += kappa * oracle.dslash(dims, WILSON, u, 1, xe)         # fills the odd half with kappa D_oe x_e
    mx = oracle.wilson_M(dims, u, kappa, full)
    mh = oracle.wilson_Mhat(dims, u, kappa, xe)
    assert rel(mx[:, :, :vh], mh[:, :, :vh]) < 1e-14
    assert np.linalg.norm(mx[:, :, vh:]) < 1e-13 * np.linalg.norm(mx)
    assert not mh[:, :, vh:].any()
    # <phi, Mhat chi> = <Mhat^+ phi, chi>
    phi = even_only(synth.source(dims, "wilson", 125), vh)
    lhs = np.vdot(phi.ravel(), mh.ravel())
    rhs = np.vdot(oracle.wilson_Mhat(dims, u, kappa, phi, dagger=True).ravel(), xe.ravel())
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4), (2, 2, 2, 2)])
def test_free_field_closed_form_of_the_preconditioned_normal_operator(dims):
    """U = 1: on the even part of a plane wave D_eo D_oe acts as D(p)^2, D(p) = 2 sum cos p - 2i sum gamma sin p,
    so Mhat^+ Mhat = 1 - 8 k^2 [(sum cos)^2 - sum sin^2] + 16 k^4 [(sum cos)^2 + sum sin^2]^2 (a scalar)."""
    kappa = 0.12
    v = synth.volume(dims)
    vh = v // 2
    u = np.broadcast_to(np.eye(3, dtype=complex), (v, 4, 3, 3)).copy()
    x = lu.site_coordinates(dims)
    rng = np.random.default_rng(3)
    for n in [(0, 0, 0, 0), (1, 0, 1, 1), (1, 1, 0, 0), tuple(rng.integers(0, 6, 4))]:
        p = lu.momenta(dims, n)
        xi = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        psi = xi[:, :, None] * np.exp(1j * (x @ p))[None, None, :]
        psi = even_only(np.ascontiguousarray(psi), vh)
        c2, s2 = np.sum(np.cos(p)) ** 2, np.sum(np.sin(p) ** 2)
        lam = 1 - 8 * kappa ** 2 * (c2 - s2) + 16 * kappa ** 4 * (c2 + s2) ** 2
        a = oracle.wilson_Mhat(dims, u, kappa, oracle.wilson_Mhat(dims, u, kappa, psi), dagger=True)
        assert rel(a, lam * psi) < 1e-13, n


def test_eo_solve_residual_and_edge_cases():
    dims, kappa = (4, 4, 4, 4), 0.12
    u = synth.gauge_field(dims, "smooth", 126)
    b = synth.source(dims, "wilson", 127)
    r = oracle.wilson_solve_eo(dims, u, kappa, 1e-10, 5000, b)
    assert r["status"] == 0
    res = rel(oracle.wilson_M(dims, u, kappa, r["x"]), b)
    assert res < 1e-9 and abs(res - r["true_residual"]) <= 1e-6 * res
    # preconditioning pays: fewer iterations than the un-preconditioned normal equations need for the same M
    plain = oracle.cg(dims, WILSON, u, kappa, 1e-10, 5000, b)
    assert r["iters"] < plain["iters"]
    z = np.zeros_like(b)
    r0 = oracle.wilson_solve_eo(dims, u, kappa, 1e-10, 10, z)
    assert r0["status"] == 0 and r0["iters"] == 0 and r0["true_residual"] == 0 and not r0["x"].any()
    r1 = oracle.wilson_solve_eo(dims, u, kappa, 1e-10, 3, b)
    assert r1["status"] == 1 and r1["iters"] == 3
