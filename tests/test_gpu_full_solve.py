"""Parity of lqcd_stag_solve_full (M x = b on the full lattice) with the
oracle's even-odd reduction, element by element on the same seeded inputs; tolerances as the CG's
(solution rel <= 1e-9 at tol 1e-10, iterations within +-2)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1311_2719_b200 import synth

pytestmark = pytest.mark.gpu

CG_TOL = 1e-9


@pytest.fixture(scope="module")
def lq():
    from paper_1311_2719_b200 import lqcd
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return lqcd


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def lattice(lq, dims, u, recon=18):
    lat = lq.Lattice(dims, lq.STAGGERED)
    lat.set_option(lq.OPT_RECONSTRUCT, recon)
    lat.load_gauge(dev(u))
    return lat


# several 128-thread tiles plus ragged tails, L = 2 (coincident neighbours), anisotropic
@pytest.mark.parametrize("dims,kind,mass", [((2, 2, 2, 2), "haar", 0.1), ((4, 4, 4, 4), "random_su3", 0.1),
                                            ((6, 4, 2, 10), "smooth", 0.05), ((10, 6, 6, 4), "haar", 0.2),
                                            ((8, 8, 8, 8), "smooth", 0.03)])
@pytest.mark.parametrize("recon", [18, 12])
def test_full_solve_matches_oracle(lq, dims, kind, mass, recon):
    u = synth.gauge_field(dims, kind, 81)
    be, bo = synth.source(dims, "staggered", 82), synth.source(dims, "staggered", 83)
    want = oracle.stag_solve_full(dims, u, mass, 1e-10, 20000, be, bo)
    assert want["status"] == 0
    with lattice(lq, dims, u, recon) as lat:
        xe, xo, it, res, status = lat.stag_solve_full(mass, 1e-10, 20000, dev(be), dev(bo))
        xe, xo = xe.cpu().numpy(), xo.cpu().numpy()
    assert status == 0 and abs(it - want["iters"]) <= 2
    assert rel(xe, want["x_e"]) <= CG_TOL
    # x_o = (b_o - D_oe x_e)/m inherits the CG's difference amplified by |D|/m, |D| <= 1/2 * 8 hops = 4
    assert rel(xo, want["x_o"]) <= CG_TOL * (4.0 / mass) * np.linalg.norm(want["x_e"]) / np.linalg.norm(want["x_o"])
    assert abs(res - want["true_residual"]) <= 0.5 * want["true_residual"] + 1e-13
    # the un-reduced system, from the oracle's bare hopping term
    me = mass * xe + oracle.dslash(dims, 0, u, 0, xo)
    mo = mass * xo + oracle.dslash(dims, 0, u, 1, xe)
    true = np.sqrt((np.linalg.norm(be - me) ** 2 + np.linalg.norm(bo - mo) ** 2) /
                   (np.linalg.norm(be) ** 2 + np.linalg.norm(bo) ** 2))
    assert abs(true - res) <= 1e-3 * true + 1e-15


def test_full_solve_fixed_iterate_and_modes(lq):
    """tol = 0: exactly k iterations, the iterate itself must agree (to rounding) with the oracle's;
    the three host-loop variants give bit-identical results."""
    c, u, _ = synth.config_inputs(2)     # 16^4 smooth
    dims, mass = c["dims"], c["param"]
    be, bo = synth.source(dims, "staggered", 84), synth.source(dims, "staggered", 85)
    want = oracle.stag_solve_full(dims, u, mass, 0.0, 9, be, bo)
    with lattice(lq, dims, u) as lat:
        got = []
        for mode in (lq.CG_SYNC, lq.CG_ASYNC, lq.CG_GRAPH):
            lat.set_option(lq.OPT_CG_MODE, mode)
            xe, xo, it, res, status = lat.stag_solve_full(mass, 0.0, 9, dev(be), dev(bo))
            got.append((xe.cpu().numpy(), xo.cpu().numpy(), it, res, status))
    xe, xo, it, res, status = got[0]
    assert status == 1 and it == 9 == want["iters"]
    assert rel(xe, want["x_e"]) <= 1e-12 and rel(xo, want["x_o"]) <= 1e-12
    assert abs(res - want["true_residual"]) <= 1e-9 * want["true_residual"]
    for other in got[1:]:
        assert np.array_equal(other[0], xe) and np.array_equal(other[1], xo) and other[2:] == (it, res, status)


def test_full_solve_edge_cases(lq):
    dims = (4, 4, 4, 4)
    u = synth.gauge_field(dims, "haar", 86)
    be, bo = synth.source(dims, "staggered", 87), synth.source(dims, "staggered", 88)
    z = np.zeros_like(be)
    with lattice(lq, dims, u) as lat:
        xe, xo, it, res, status = lat.stag_solve_full(0.1, 1e-10, 100, dev(z), dev(z))
        assert it == 0 and res == 0.0 and status == 0 and not xe.any().item() and not xo.any().item()
        # odd-site source only
        want = oracle.stag_solve_full(dims, u, 0.1, 1e-10, 5000, z, bo)
        xe, xo, it, res, status = lat.stag_solve_full(0.1, 1e-10, 5000, dev(z), dev(bo))
        assert status == 0 and abs(it - want["iters"]) <= 2
        assert rel(xe.cpu().numpy(), want["x_e"]) <= CG_TOL and rel(xo.cpu().numpy(), want["x_o"]) <= CG_TOL * 4.0 / 0.1
        bed, bod = dev(be), dev(bo)
        with pytest.raises(lq.LqcdError):
            lat.stag_solve_full(0.0, 1e-10, 10, bed, bod)                 # mass = 0
        with pytest.raises(lq.LqcdError):
            lat.stag_solve_full(0.1, 1e-10, 10, bed, bod, bed, None)      # aliasing
        xe, xo, it, res, status = lat.stag_solve_full(0.1, 1e-10, 3, bed, bod)
        assert it == 3 and status == 1
    uw = synth.gauge_field(dims, "smooth", 89)
    with lq.Lattice(dims, lq.WILSON) as wl:
        wl.load_gauge(dev(uw))
        with pytest.raises((lq.LqcdError, ValueError)):
            wl.stag_solve_full(0.1, 1e-10, 10, bed, bod)


@pytest.mark.slow
def test_full_solve_cfg3_properties(lq):
    """Full size (32^4 Haar, m = 0.01) in the bench's launch configuration: the un-reduced residual
    from sampled oracle Dslash sites and the norm identity |b - M x| = |b' - A x_e| / m."""
    c, u, _ = synth.config_inputs(3)
    dims, mass = c["dims"], c["param"]
    be, bo = synth.source(dims, "staggered", 90), synth.source(dims, "staggered", 91)
    with lattice(lq, dims, u) as lat:
        lat.set_option(lq.OPT_CG_MODE, lq.CG_GRAPH)
        lat.set_option(lq.OPT_CG_CHECK_EVERY, 8)
        xe, xo, it, res, status = lat.stag_solve_full(mass, 1e-10, 100000, dev(be), dev(bo))
        xe, xo = xe.cpu().numpy(), xo.cpu().numpy()
    assert status == 0
    rng = np.random.default_rng(5)
    e = rng.integers(0, be.shape[1], 4096)
    me = mass * xe[:, e].T + oracle.dslash_sites(dims, 0, u, 0, xo, e)
    mo = mass * xo[:, e].T + oracle.dslash_sites(dims, 0, u, 1, xe, e)
    scale = np.sqrt((np.linalg.norm(be) ** 2 + np.linalg.norm(bo) ** 2) / (2 * be.size))   # rms |b_i|
    assert np.abs(be[:, e].T - me).max() <= 1e-6 * scale     # |r_i| <~ |r'|_inf / m, tol 1e-10 / m = 1e-8
    assert np.abs(bo[:, e].T - mo).max() <= 1e-9 * scale     # the odd rows hold to rounding by construction
    assert res <= 1e-10 * (mass + 4.0) / mass
