"""Pins for the CPU oracle (BASELINE.json north_star): what the
mathematics fixes, never the oracle against itself.  No GPU needed.

P1 free staggered spectrum   P2 anti-hermiticity of D     P3 hermiticity/positivity of M^+M
P4 gauge covariance          P5 gamma5-hermiticity        P6 free Wilson spectrum
P7 dense inversion on 2^4    P8 neighbour tables          P9 CG recursion vs true residual
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from oracle import STAGGERED, WILSON, EVEN, ODD
from paper_1311_2719_b200 import synth

import lattice_util as lu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")

SHAPES = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4), (6, 4, 2, 2), (2, 4, 4, 8)]


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


# ---------------------------------------------------------------- P8 tables

@pytest.mark.parametrize("dims", SHAPES + [(16, 16, 16, 16), (16, 16, 16, 32)])
def test_tables_match_independent_coordinate_arithmetic(dims):
    iup, idn, l2e = oracle.tables(dims)
    v = synth.volume(dims)
    vh = v // 2
    assert iup.dtype == np.int32 and iup.shape == (4, v)
    x = lu.site_coordinates(dims)
    assert np.array_equal(oracle.coords(dims), x)
    for mu in range(4):
        assert np.array_equal(iup[mu], lu.shifted_index(dims, mu, +1))
        assert np.array_equal(idn[mu], lu.shifted_index(dims, mu, -1))
        # permutations, inverse of each other, mapping parity p onto 1-p
        assert np.array_equal(np.sort(iup[mu]), np.arange(v))
        assert np.array_equal(idn[mu][iup[mu]], np.arange(v))
        assert np.all((iup[mu][:vh] >= vh)) and np.all((iup[mu][vh:] < vh))
    # lex2eo: s -> g
    s = x[:, 0] + dims[0] * (x[:, 1] + dims[1] * (x[:, 2] + dims[2] * x[:, 3]))
    assert np.array_equal(l2e[s], np.arange(v))


def test_half_index_neighbours_in_fastest_dimension():
    # SURVEY 8(c.1) consequence: +x0 neighbour of half-index e is e (x0 even) or e+1 (x0 odd, wrapping in the row)
    dims = (8, 4, 4, 4)
    iup, idn, _ = oracle.tables(dims)
    v = synth.volume(dims)
    vh, lh = v // 2, dims[0] // 2
    x = lu.site_coordinates(dims)
    e = np.arange(v) % vh
    up_e = iup[0] % vh
    row0 = (e // lh) * lh
    expect = np.where(x[:, 0] % 2 == 0, e, row0 + (e - row0 + 1) % lh)
    assert np.array_equal(up_e, expect)


def test_odd_or_small_extent_is_an_error():
    with pytest.raises(ValueError):
        oracle.tables((3, 4, 4, 4))
    with pytest.raises(ValueError):
        oracle.tables((4, 4, 4, 0))


# ------------------------------------------------- P1 free staggered spectrum

def plane_wave(dims, p, x):
    return np.exp(1j * (x @ p))


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4), (2, 2, 2, 2), (6, 4, 2, 8)])
def test_free_staggered_spectrum(dims):
    """U = 1: A chi = (m^2 + sum_mu sin^2 p_mu) chi for chi = e^{ipx} c on even sites,
    p_3 half-integer (antiperiodic time).  Catches a missing 1/2, wrong eta phases
    (eta = 1 would give (sum sin p)^2), a periodic time boundary, a wrong mass term."""
    u = synth.gauge_field(dims, "unit", 0)
    v = synth.volume(dims)
    vh = v // 2
    x = lu.site_coordinates(dims)[:vh].astype(np.float64)
    m = 0.37
    rng = np.random.default_rng(5)
    all_n = list(itertools.product(*[range(L) for L in dims]))
    pick = all_n if len(all_n) <= 64 else [all_n[i] for i in rng.choice(len(all_n), 48, replace=False)]
    for n in pick:
        p = lu.momenta(dims, n)
        c = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        chi = c[:, None] * plane_wave(dims, p, x)[None, :]
        lam = m * m + np.sum(np.sin(p) ** 2)
        out = oracle.apply_MdagM(dims, STAGGERED, u, m, chi)
        assert rel(out, lam * chi) < 1e-13, (n, lam)
    # integer time momentum must NOT be an eigenvector (the boundary is antiperiodic).  Only
    # meaningful for L3 > 4: at L3 = 4 (and 2) every half-integer mode has the same sin^2 p_3,
    # so the time part of -D^2 is a multiple of the identity.
    if dims[3] > 4:
        p = 2 * np.pi * np.array([1, 0, 0, 1]) / np.array(dims)
        chi = np.ones(3)[:, None] * plane_wave(dims, p, x)[None, :]
        out = oracle.apply_MdagM(dims, STAGGERED, u, m, chi)
        lam = vdot(chi, out) / vdot(chi, chi)
        assert rel(out, lam * chi) > 1e-3


def test_free_staggered_D_squared_on_odd_sites_too():
    # -D_oe D_eo on the odd sublattice has the same free spectrum
    dims = (4, 4, 2, 4)
    u = synth.gauge_field(dims, "unit", 0)
    vh = synth.volume(dims) // 2
    x = lu.site_coordinates(dims)[vh:].astype(np.float64)
    p = lu.momenta(dims, (1, 3, 1, 2))
    chi = np.array([1.0, -2.0j, 0.5])[:, None] * plane_wave(dims, p, x)[None, :]
    t = oracle.dslash(dims, STAGGERED, u, EVEN, chi)
    out = -oracle.dslash(dims, STAGGERED, u, ODD, t)
    assert rel(out, np.sum(np.sin(p) ** 2) * chi) < 1e-13


# --------------------------------------------- P2 / P3 (anti-)hermiticity

@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("kind", ["haar", "smooth"])
def test_staggered_antihermitian_and_MdagM_hermitian_positive(dims, kind):
    u = synth.gauge_field(dims, kind, 11)
    vh = synth.volume(dims) // 2
    chi = synth.vector((3, vh), 1)
    phi_o = synth.vector((3, vh), 2)
    phi = synth.vector((3, vh), 3)
    d_chi = oracle.dslash(dims, STAGGERED, u, ODD, chi)     # D_oe chi_e
    d_phi = oracle.dslash(dims, STAGGERED, u, EVEN, phi_o)  # D_eo phi_o
    lhs, rhs = vdot(phi_o, d_chi), -vdot(d_phi, chi)
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)
    m = 0.1
    a_chi = oracle.apply_MdagM(dims, STAGGERED, u, m, chi)
    a_phi = oracle.apply_MdagM(dims, STAGGERED, u, m, phi)
    assert abs(vdot(phi, a_chi) - vdot(a_phi, chi)) < 1e-13 * abs(vdot(phi, a_chi))
    q = vdot(chi, a_chi)
    expect = m * m * vdot(chi, chi).real + vdot(d_chi, d_chi).real   # PAPER.md:85, <p,Ap> from norms only
    assert abs(q.imag) < 1e-13 * abs(q.real)                          # reading A9
    assert abs(q.real - expect) < 1e-13 * expect
    assert q.real >= m * m * vdot(chi, chi).real


# ------------------------------------------------------ P4 gauge covariance

def gauge_transform(dims, u, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^+ with the test's own neighbour arithmetic."""
    out = np.empty_like(u)
    for mu in range(4):
        up = lu.shifted_index(dims, mu, +1)
        out[:, mu] = g @ u[:, mu] @ np.conj(np.swapaxes(g[up], 1, 2))
    return out


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (4, 2, 6, 4)])
def test_gauge_covariance_staggered(dims):
    v = synth.volume(dims)
    vh = v // 2
    u = synth.gauge_field(dims, "haar", 21)
    g = synth.su3_field(v, 22)
    u2 = gauge_transform(dims, u, g)
    for out_parity in (EVEN, ODD):
        gin = g[vh:] if out_parity == EVEN else g[:vh]
        gout = g[:vh] if out_parity == EVEN else g[vh:]
        chi = synth.vector((3, vh), 23 + out_parity)
        chi2 = np.einsum("eab,be->ae", gin, chi)
        lhs = oracle.dslash(dims, STAGGERED, u2, out_parity, chi2)
        rhs = np.einsum("eab,be->ae", gout, oracle.dslash(dims, STAGGERED, u, out_parity, chi))
        assert rel(lhs, rhs) < 1e-13
        # and a transposed / conjugated link must break it (the test has teeth)
        bad = oracle.dslash(dims, STAGGERED, np.swapaxes(u2, 2, 3), out_parity, chi2)
        assert rel(bad, rhs) > 1e-2


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (4, 2, 6, 4)])
def test_gauge_covariance_wilson(dims):
    v = synth.volume(dims)
    u = synth.gauge_field(dims, "haar", 31)
    g = synth.su3_field(v, 32)
    u2 = gauge_transform(dims, u, g)
    psi = synth.vector((4, 3, v), 33)
    psi2 = np.einsum("gab,sbg->sag", g, psi)
    for out_parity in (EVEN, ODD):
        lhs = oracle.dslash(dims, WILSON, u2, out_parity, psi2)
        rhs = np.einsum("gab,sbg->sag", g, oracle.dslash(dims, WILSON, u, out_parity, psi))
        assert rel(lhs, rhs) < 1e-13
    kappa = 0.12
    lhs = oracle.apply_MdagM(dims, WILSON, u2, kappa, psi2)
    rhs = np.einsum("gab,sbg->sag", g, oracle.apply_MdagM(dims, WILSON, u, kappa, psi))
    assert rel(lhs, rhs) < 1e-13


# --------------------------------------------------- P5 gamma5-hermiticity

@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (2, 4, 4, 8)])
def test_wilson_gamma5_hermiticity(dims):
    v = synth.volume(dims)
    u = synth.gauge_field(dims, "haar", 41)
    phi = synth.vector((4, 3, v), 42)
    psi = synth.vector((4, 3, v), 43)
    g5 = np.array([1, 1, -1, -1.0])[:, None, None]
    kappa = 0.12
    lhs = vdot(phi, oracle.wilson_M(dims, u, kappa, psi))
    rhs = vdot(g5 * oracle.wilson_M(dims, u, kappa, g5 * phi), psi)
    assert abs(lhs - rhs) < 1e-13 * abs(lhs)
    # M^+M as returned = gamma5 M gamma5 M, hermitian, <psi,A psi> = |M psi|^2
    a_psi = oracle.apply_MdagM(dims, WILSON, u, kappa, psi)
    a_phi = oracle.apply_MdagM(dims, WILSON, u, kappa, phi)
    assert abs(vdot(phi, a_psi) - vdot(a_phi, psi)) < 1e-13 * abs(vdot(phi, a_psi))
    m_psi = oracle.wilson_M(dims, u, kappa, psi)
    assert abs(vdot(psi, a_psi) - vdot(m_psi, m_psi)) < 1e-13 * abs(vdot(m_psi, m_psi))
    # the hopping term alone: gamma5 D gamma5 = D^+
    d_psi = oracle.dslash(dims, WILSON, u, EVEN, psi) + oracle.dslash(dims, WILSON, u, ODD, psi)
    d_phi = oracle.dslash(dims, WILSON, u, EVEN, g5 * phi) + oracle.dslash(dims, WILSON, u, ODD, g5 * phi)
    assert abs(vdot(phi, d_psi) - vdot(g5 * d_phi, psi)) < 1e-13 * abs(vdot(phi, d_psi))


# ----------------------------------------------------- P6 free Wilson spectrum

@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 2, 6, 4), (2, 2, 2, 2)])
def test_free_wilson_spectrum_and_gamma_basis(dims):
    """U = 1: M e^{ipx} xi = e^{ipx} [1 - 2k sum cos p + 2ik sum gamma_mu sin p_mu] xi with the
    DeGrand-Rossi matrices of tests/golden, hence A e^{ipx} xi = [(1-2k sum cos)^2 + 4k^2 sum sin^2] e^{ipx} xi."""
    gam = lu.read_gammas(os.path.join(GOLDEN, "degrand_rossi_gamma.txt"))
    for mu in range(4):       # the fixture itself: hermitian Clifford algebra, gamma5 = diag(1,1,-1,-1)
        assert np.allclose(gam[mu], gam[mu].conj().T)
        for nu in range(4):
            assert np.allclose(gam[mu] @ gam[nu] + gam[nu] @ gam[mu], 2 * np.eye(4) * (mu == nu))
    assert np.allclose(gam[0] @ gam[1] @ gam[2] @ gam[3], np.diag([1, 1, -1, -1]))
    u = synth.gauge_field(dims, "unit", 0)
    x = lu.site_coordinates(dims).astype(np.float64)
    kappa = 0.12
    rng = np.random.default_rng(6)
    all_n = list(itertools.product(*[range(L) for L in dims]))
    pick = all_n if len(all_n) <= 16 else [all_n[i] for i in rng.choice(len(all_n), 16, replace=False)]
    for n in pick:
        p = lu.momenta(dims, n)
        xi = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi = xi[:, :, None] * plane_wave(dims, p, x)[None, None, :]
        mp = (1 - 2 * kappa * np.sum(np.cos(p))) * np.eye(4) + 2j * kappa * np.einsum("m,mst->st", np.sin(p), gam)
        expect_m = np.einsum("st,tc->sc", mp, xi)[:, :, None] * plane_wave(dims, p, x)[None, None, :]
        assert rel(oracle.wilson_M(dims, u, kappa, psi), expect_m) < 1e-13, n
        lam = (1 - 2 * kappa * np.sum(np.cos(p))) ** 2 + 4 * kappa ** 2 * np.sum(np.sin(p) ** 2)
        assert rel(oracle.apply_MdagM(dims, WILSON, u, kappa, psi), lam * psi) < 1e-13, n


# ------------------------------------------------- P7 dense inversion on 2^4

def dense_matrix(apply, shape):
    n = int(np.prod(shape))
    a = np.empty((n, n), complex)
    for j in range(n):
        e = np.zeros(n, complex)
        e[j] = 1.0
        a[:, j] = apply(e.reshape(shape)).ravel()
    return a


@pytest.mark.parametrize("fermion,param,kind", [(STAGGERED, 0.1, "haar"), (STAGGERED, 0.05, "smooth"),
                                                (WILSON, 0.12, "smooth"), (WILSON, 0.1, "haar")])
def test_cg_against_dense_solve_on_2_4(fermion, param, kind):
    dims = (2, 2, 2, 2)
    u = synth.gauge_field(dims, kind, 51)
    b = synth.source(dims, "staggered" if fermion == STAGGERED else "wilson", 52)
    a = dense_matrix(lambda v: oracle.apply_MdagM(dims, fermion, u, param, v), b.shape)
    assert np.allclose(a, a.conj().T, atol=1e-14)
    w = np.linalg.eigvalsh(a)
    if fermion == STAGGERED:
        assert w.min() >= param ** 2 * (1 - 1e-12)
    else:
        assert w.min() > 0
    x_dense = np.linalg.solve(a, b.ravel()).reshape(b.shape)
    r = oracle.cg(dims, fermion, u, param, 1e-12, 1000, b)
    assert r["status"] == 0
    assert rel(r["x"], x_dense) < 1e-9
    # exact-arithmetic CG ends in at most n steps (number of distinct eigenvalues); allow rounding slack
    assert r["iters"] <= b.size + 10
    assert r["true_residual"] < 1e-11


def test_cg_zero_source_and_maxiter():
    dims = (2, 2, 2, 2)
    u = synth.gauge_field(dims, "haar", 61)
    b = np.zeros((3, 8), complex)
    r = oracle.cg(dims, STAGGERED, u, 0.1, 1e-10, 10, b)
    assert r["iters"] == 0 and r["status"] == 0 and r["true_residual"] == 0 and not r["x"].any()
    b = synth.source((4, 4, 4, 4), "staggered", 62)
    u = synth.gauge_field((4, 4, 4, 4), "haar", 63)
    r = oracle.cg((4, 4, 4, 4), STAGGERED, u, 0.01, 1e-10, 7, b)
    assert r["status"] == 1 and r["iters"] == 7
    # tol = 0: exactly maxiter iterations
    r0 = oracle.cg((4, 4, 4, 4), STAGGERED, u, 0.01, 0.0, 7, b)
    assert r0["status"] == 1 and r0["iters"] == 7 and np.array_equal(r0["x"], r["x"])


# --------------------------------------------------------- P9 CG sanity

def test_cg_recursion_residual_matches_true_residual_cfg1():
    c, u, b = synth.config_inputs(1)
    r = oracle.cg(c["dims"], STAGGERED, u, c["param"], c["tol"], 5000, b, history=True)
    assert r["status"] == 0
    h = r["rr_history"]
    assert len(h) == r["iters"] + 1
    bb = vdot(b, b).real
    assert abs(h[0] - bb) < 1e-12 * bb
    assert h[-1] <= c["tol"] ** 2 * bb < h[-2]
    rec = np.sqrt(h[-1] / bb)
    assert abs(rec - r["true_residual"]) < 1e-3 * r["true_residual"] and r["true_residual"] < 2e-10
    # the solution satisfies the equation as checked with numpy on the oracle's operator output
    ax = oracle.apply_MdagM(c["dims"], STAGGERED, u, c["param"], r["x"])
    assert rel(ax, b) < 2e-10


@pytest.mark.parametrize("fermion", [STAGGERED, WILSON])
def test_cg_true_residual_is_the_fresh_residual(fermion):
    """`true_residual` is |b - A x| / |b| with a FRESH application of A (SURVEY 8(c.4) last line; the
    exit test itself, uses the recursion's <r,r>).  The norm is retaken here in numpy
    from the oracle's operator output; the two agree to summation-order rounding (1e-12 relative), while
    the recursion's value is measurably different after a few hundred iterations -- so a residual
    reported from the recursion, a missing sqrt, or a division by <r,r> instead of <b,b> fails."""
    if fermion == STAGGERED:
        c, u, b = synth.config_inputs(1)
        dims, param = c["dims"], c["param"]
    else:
        dims, param = (4, 4, 4, 4), 0.12
        u = synth.gauge_field(dims, "smooth", 5)
        b = synth.source(dims, "wilson", 6)
    r = oracle.cg(dims, fermion, u, param, 1e-10, 5000, b, history=True)
    assert r["status"] == 0
    ax = oracle.apply_MdagM(dims, fermion, u, param, r["x"])
    fresh = np.linalg.norm((b - ax).ravel()) / np.linalg.norm(b.ravel())
    assert abs(fresh - r["true_residual"]) <= 1e-12 * fresh
    rec = np.sqrt(r["rr_history"][-1] / vdot(b, b).real)
    assert abs(rec - fresh) > 1e-8 * fresh        # the pin above can tell the two apart ...
    assert abs(rec - fresh) < 1e-3 * fresh        # ... and the recursion has not drifted (P9)
    # a MAXITER exit reports the residual of the iterate it returns, not of a converged one
    r7 = oracle.cg(dims, fermion, u, param, 1e-10, 7, b)
    ax7 = oracle.apply_MdagM(dims, fermion, u, param, r7["x"])
    fresh7 = np.linalg.norm((b - ax7).ravel()) / np.linalg.norm(b.ravel())
    assert r7["status"] == 1 and fresh7 > 1e-3 and abs(fresh7 - r7["true_residual"]) <= 1e-12 * fresh7


def test_dot_re_over_several_blocks_and_a_ragged_tail():
    """oracle.dot_re sums in fixed 4096-element blocks; n = 3 blocks + 17 exercises the block loop and
    the tail (a dropped tail block or a wrong block bound changes the sum by O(1))."""
    rng = np.random.default_rng(1311)
    for n in (1, 17, 4096, 4097, 3 * 4096 + 17):
        a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
        want = np.vdot(a, b).real
        scale = np.linalg.norm(a) * np.linalg.norm(b)
        assert abs(oracle.dot_re(a, b) - want) <= 1e-14 * scale
        assert abs(oracle.dot_re(a, a) - np.linalg.norm(a) ** 2) <= 1e-14 * scale
    # Re<a,b> = Re conj(a).b: conjugation on the FIRST argument, real part only
    a = np.array([1 + 2j, 3 - 1j]); b = np.array([2 - 1j, 1j])
    assert oracle.dot_re(a, b) == (np.conj(a) * b).sum().real == -1.0


@pytest.mark.parametrize("cfg", [1, 2])
def test_thread_count_does_not_change_results(cfg):
    """cfg 1: 384 elements = one block of the blocked dot product; cfg 2: 98 304 elements = 24 blocks
    shared out between the threads -- the path every 16^4 and larger CG takes."""
    c, u, b = synth.config_inputs(cfg)
    n0 = oracle.num_threads()
    try:
        oracle.set_threads(1)
        r1 = oracle.cg(c["dims"], STAGGERED, u, c["param"], c["tol"], 5000, b)
        oracle.set_threads(max(2, n0))
        r2 = oracle.cg(c["dims"], STAGGERED, u, c["param"], c["tol"], 5000, b)
    finally:
        oracle.set_threads(n0)
    assert r1["iters"] == r2["iters"] and np.array_equal(r1["x"], r2["x"])


def test_dslash_sites_equals_full_dslash():
    dims = (4, 2, 6, 4)
    v = synth.volume(dims)
    u = synth.gauge_field(dims, "smooth", 71)
    e = np.array([0, 1, 5, v // 2 - 1, 17])
    chi = synth.vector((3, v // 2), 72)
    for par in (EVEN, ODD):
        full = oracle.dslash(dims, STAGGERED, u, par, chi)
        assert np.array_equal(oracle.dslash_sites(dims, STAGGERED, u, par, chi, e), full[:, e].T)
    psi = synth.vector((4, 3, v), 73)
    for par in (EVEN, ODD):
        full = oracle.dslash(dims, WILSON, u, par, psi)
        got = oracle.dslash_sites(dims, WILSON, u, par, psi, e)
        assert np.array_equal(got, np.moveaxis(full[:, :, par * (v // 2) + e], 2, 0))


# --------------------------------------------------- input recipe (A18)

@pytest.mark.parametrize("kind", ["random_su3", "smooth", "haar"])
def test_links_are_su3(kind):
    u = synth.gauge_field((4, 4, 4, 4), kind, 81).reshape(-1, 3, 3)
    assert np.abs(u @ np.conj(np.swapaxes(u, 1, 2)) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(u) - 1).max() < 1e-14
    if kind == "smooth":   # close to the identity: |U - 1| of order eps
        assert 0.05 < np.abs(u - np.eye(3)).mean() < 0.3


def test_generators_are_reproducible_and_thread_independent():
    a = synth.gauge_field((8, 8, 8, 8), "haar", 3, threads=1)
    b = synth.gauge_field((8, 8, 8, 8), "haar", 3, threads=4)
    assert np.array_equal(a, b)
    assert not np.array_equal(a, synth.gauge_field((8, 8, 8, 8), "haar", 4))
    assert np.array_equal(synth.source((4, 4, 4, 4), "wilson", 9), synth.source((4, 4, 4, 4), "wilson", 9))
