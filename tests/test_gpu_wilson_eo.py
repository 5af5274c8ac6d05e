"""Parity of the even-odd preconditioned Wilson solver (lqcd_wilson_eo_MdagM, lqcd_wilson_solve_eo;
SURVEY.md 8(f) row 4) with the oracle, element by element on the same seeded inputs.  Tolerances as the
north star's: operator rel-L2 <= 1e-13, solution rel <= 1e-9 at tol 1e-10, iterations within +-2."""
import numpy as np
import pytest
import torch

import oracle
from paper_1311_2719_b200 import synth

pytestmark = pytest.mark.gpu

SHAPES = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 8), (6, 4, 2, 2), (10, 6, 6, 4), (8, 8, 8, 8)]


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
    lat = lq.Lattice(dims, lq.WILSON)
    lat.set_option(lq.OPT_RECONSTRUCT, recon)
    lat.load_gauge(dev(u))
    return lat


@pytest.mark.parametrize("dims", SHAPES)
@pytest.mark.parametrize("recon", [18, 12])
def test_eo_normal_operator(lq, dims, recon):
    kappa = 0.12
    vh = synth.volume(dims) // 2
    u = synth.gauge_field(dims, "haar", 131)
    v = synth.source(dims, "wilson", 132)
    want = oracle.wilson_Mhat(dims, u, kappa, oracle.wilson_Mhat(dims, u, kappa, v), dagger=True)
    with lattice(lq, dims, u, recon) as lat:
        sentinel = torch.full(lat.vector_shape, 7.0 + 0j, dtype=torch.complex128, device="cuda")
        got = lat.wilson_eo_MdagM(kappa, dev(v), sentinel).cpu().numpy()
    assert rel(got[:, :, :vh], want[:, :, :vh]) <= 1e-13
    assert np.all(got[:, :, vh:] == 7.0)           # the odd half is not written


@pytest.mark.parametrize("dims,kind,kappa", [((2, 2, 2, 2), "smooth", 0.12), ((4, 4, 4, 4), "haar", 0.1),
                                             ((4, 2, 6, 8), "smooth", 0.12), ((10, 6, 6, 4), "random_su3", 0.09),
                                             ((8, 8, 8, 8), "smooth", 0.125)])
@pytest.mark.parametrize("recon", [18, 12])
def test_eo_solve_matches_oracle(lq, dims, kind, kappa, recon):
    u = synth.gauge_field(dims, kind, 133)
    b = synth.source(dims, "wilson", 134)
    want = oracle.wilson_solve_eo(dims, u, kappa, 1e-10, 20000, b)
    assert want["status"] == 0
    with lattice(lq, dims, u, recon) as lat:
        x, it, res, status = lat.wilson_solve_eo(kappa, 1e-10, 20000, dev(b))
        x = x.cpu().numpy()
    assert status == 0 and abs(it - want["iters"]) <= 2
    assert rel(x, want["x"]) <= 1e-9
    true = rel(oracle.wilson_M(dims, u, kappa, x), b)      # the un-reduced system, oracle's full-lattice M
    assert abs(true - res) <= 1e-3 * true + 1e-15
    assert abs(res - want["true_residual"]) <= 0.5 * want["true_residual"] + 1e-13


def test_eo_solve_cfg4_modes_and_iteration_gain(lq):
    """BASELINE config 4 (16^3x32, kappa 0.12): the three host-loop variants agree bit for bit, and the
    preconditioned solve of M x = b needs fewer iterations than config 4's CG on M^+M."""
    c, u, b = synth.config_inputs(4)
    dims, kappa = c["dims"], c["param"]
    want = oracle.wilson_solve_eo(dims, u, kappa, 1e-10, 20000, b)
    with lattice(lq, dims, u) as lat:
        got = []
        for mode in (lq.CG_SYNC, lq.CG_ASYNC, lq.CG_GRAPH):
            lat.set_option(lq.OPT_CG_MODE, mode)
            x, it, res, status = lat.wilson_solve_eo(kappa, 1e-10, 20000, dev(b))
            got.append((x.cpu().numpy(), it, res, status))
        _, it_full, _, _ = lat.cg_solve(kappa, 1e-10, 20000, dev(b))
    x, it, res, status = got[0]
    assert status == 0 and abs(it - want["iters"]) <= 2 and rel(x, want["x"]) <= 1e-9
    for other in got[1:]:
        assert np.array_equal(other[0], x) and other[1:] == (it, res, status)
    assert it < it_full


def test_eo_solve_edge_cases(lq):
    dims, kappa = (4, 4, 4, 4), 0.12
    u = synth.gauge_field(dims, "smooth", 135)
    b = synth.source(dims, "wilson", 136)
    with lattice(lq, dims, u) as lat:
        z = torch.zeros_like(dev(b))
        x, it, res, status = lat.wilson_solve_eo(kappa, 1e-10, 100, z)
        assert (it, res, status) == (0, 0.0, 0) and not x.any().item()
        for k in (1, 4):
            want = oracle.wilson_solve_eo(dims, u, kappa, 0.0, k, b)
            x, it, res, status = lat.wilson_solve_eo(kappa, 0.0, k, dev(b))
            assert status == 1 and it == k and rel(x.cpu().numpy(), want["x"]) <= 1e-12
            assert abs(res - want["true_residual"]) <= 1e-9 * want["true_residual"]
        bd = dev(b)
        with pytest.raises(lq.LqcdError):
            lat.wilson_solve_eo(kappa, 1e-10, 10, bd, bd)
    us = synth.gauge_field(dims, "haar", 137)
    with lq.Lattice(dims, lq.STAGGERED) as sl:
        sl.load_gauge(dev(us))
        bs = dev(synth.source(dims, "staggered", 138))
        with pytest.raises(lq.LqcdError):
            sl.wilson_solve_eo(kappa, 1e-10, 10, bs)
        with pytest.raises(lq.LqcdError):
            sl.wilson_eo_MdagM(kappa, bs)
