"""Parity of lqcd_cg_solve_mixed (fp32 inner CG + fp64 reliable updates) with
the oracle's mixed-precision CG and with the plain fp64 solution.

Contract: the exit is declared on an fp64 residual, so true_residual
<= tol; the solution agrees with the fp64 CG's within the bound two tol-converged solutions obey,
2 tol |b| / (m^2 |x|) (and within 1e-8 here); fp32 rounding perturbs the trajectory, so iteration
and update counts are compared with the oracle's mixed solver within a few per cent, not +-2; the
first iterates (before rounding has separated the two) agree to fp32 accuracy."""

import numpy as np
import pytest
import torch

import oracle
from paper_1311_2719_b200 import synth
from lattice_util import check_sampled_solution, golden

pytestmark = pytest.mark.gpu


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


def count_close(a, b):
    return abs(a - b) <= max(3, 0.03 * b)


@pytest.mark.parametrize("dims,kind,mass", [((2, 2, 2, 2), "haar", 0.1), ((4, 4, 4, 4), "random_su3", 0.1),
                                            ((6, 4, 2, 10), "smooth", 0.05), ((10, 6, 6, 4), "haar", 0.2),
                                            ((8, 8, 8, 8), "haar", 0.03), ((16, 16, 16, 16), "smooth", 0.05)])
@pytest.mark.parametrize("recon", [18, 12])
def test_mixed_cg_matches_oracle(lq, dims, kind, mass, recon):
    tol = 1e-10
    u = synth.gauge_field(dims, kind, 111)
    b = synth.source(dims, "staggered", 112)
    want = oracle.cg_mixed(dims, u, mass, tol, 20000, b, history=True)
    plain = oracle.cg(dims, 0, u, mass, tol, 20000, b)
    assert want["status"] == 0
    with lattice(lq, dims, u, recon) as lat:
        x, it, nupd, res, status = lat.cg_solve_mixed(mass, tol, 20000, dev(b))
        x = x.cpu().numpy()
        hist = lat.cg_history().numpy()
    assert status == 0 and res <= tol
    bound = 2 * tol * np.linalg.norm(b) / mass ** 2
    assert np.linalg.norm(x - plain["x"]) <= min(bound, 1e-8 * np.linalg.norm(plain["x"]))
    assert np.linalg.norm(x - want["x"]) <= min(bound, 1e-8 * np.linalg.norm(want["x"]))
    assert count_close(it, want["iters"]) and abs(nupd - want["updates"]) <= 2
    # residual from its definition, with the oracle's fp64 operator
    true = rel(oracle.apply_MdagM(dims, 0, u, mass, x), b)
    assert abs(true - res) <= 1e-3 * true + 1e-15
    # the first iterations follow the oracle's to fp32 accuracy
    n = min(len(hist), len(want["rr_history"]), 6)
    assert np.allclose(hist[:n], want["rr_history"][:n], rtol=2e-5)


def test_mixed_cg_modes_and_batching_give_identical_results(lq):
    c, u, b = synth.config_inputs(1)
    with lattice(lq, c["dims"], u) as lat:
        lat.set_option(lq.OPT_CG_MODE, lq.CG_SYNC)
        x0, it0, n0, res0, st0 = lat.cg_solve_mixed(c["param"], c["tol"], 20000, dev(b))
        h0 = lat.cg_history().numpy()
        x0 = x0.cpu().numpy()
        for mode, every in ((lq.CG_ASYNC, 1), (lq.CG_ASYNC, 5), (lq.CG_GRAPH, 8), (lq.CG_GRAPH, 16)):
            lat.set_option(lq.OPT_CG_MODE, mode)
            lat.set_option(lq.OPT_CG_CHECK_EVERY, every)
            x1, it1, n1, res1, st1 = lat.cg_solve_mixed(c["param"], c["tol"], 20000, dev(b))
            assert (it1, n1, res1, st1) == (it0, n0, res0, st0) and np.array_equal(x1.cpu().numpy(), x0)
            assert np.array_equal(lat.cg_history().numpy(), h0)
        # and the fp64 solver on the same context is not disturbed by the mixed one's state
        want = oracle.cg(c["dims"], 0, u, c["param"], c["tol"], 20000, b)
        x, it, res, status = lat.cg_solve(c["param"], c["tol"], 20000, dev(b))
        assert status == 0 and abs(it - want["iters"]) <= 2 and rel(x.cpu().numpy(), want["x"]) <= 1e-9


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (8, 4, 6, 2), (12, 2, 2, 4), (4, 6, 10, 8), (16, 16, 16, 16)])
def test_mixed_cg_two_sites_per_thread_kernels(lq, dims, recon):
    """LQCD_OPT_F32_PAIRS (default on where L0 % 4 == 0): two sites per thread with 128-bit loads.  Same
    per-site arithmetic as the one-site kernels -- only the partial sums are grouped differently, so
    fixed-iteration iterates agree far below fp32 accuracy -- and the same parity with the oracle."""
    mass = 0.08
    u = synth.gauge_field(dims, "haar", 211)
    b = synth.source(dims, "staggered", 212)
    with lattice(lq, dims, u, recon) as lat:
        for k in (1, 7):
            got = []
            for pairs in (1, 0):
                lat.set_option(lq.OPT_F32_PAIRS, pairs)
                x, it, nupd, res, status = lat.cg_solve_mixed(mass, 0.0, k, dev(b))
                got.append((x.cpu().numpy(), it, lat.cg_history().numpy()))
            assert got[0][1] == got[1][1] == k
            assert rel(got[0][0], got[1][0]) <= 1e-6
            assert np.allclose(got[0][2], got[1][2], rtol=1e-6)
            want = oracle.cg_mixed(dims, u, mass, 0.0, k, b)
            assert rel(got[0][0], want["x"]) <= 2e-5
        lat.set_option(lq.OPT_F32_PAIRS, 1)
        want = oracle.cg_mixed(dims, u, mass, 1e-10, 20000, b)
        x, it, nupd, res, status = lat.cg_solve_mixed(mass, 1e-10, 20000, dev(b))
        assert status == 0 and res <= 1e-10 and count_close(it, want["iters"]) and abs(nupd - want["updates"]) <= 2
        assert np.linalg.norm(x.cpu().numpy() - want["x"]) <= 1e-8 * np.linalg.norm(want["x"])


def test_mixed_cg_fixed_iterations_and_edge_cases(lq):
    dims, mass = (8, 8, 8, 4), 0.1
    u = synth.gauge_field(dims, "haar", 113)
    b = synth.source(dims, "staggered", 114)
    with lattice(lq, dims, u) as lat:
        for k in (1, 5, 40):
            want = oracle.cg_mixed(dims, u, mass, 0.0, k, b)
            x, it, nupd, res, status = lat.cg_solve_mixed(mass, 0.0, k, dev(b))
            assert status == 1 and it == k == want["iters"] and abs(nupd - want["updates"]) <= 1
            assert rel(x.cpu().numpy(), want["x"]) <= 2e-5          # iterates agree to fp32 accuracy
            assert abs(res - want["true_residual"]) <= 1e-3 * want["true_residual"]
        z = torch.zeros_like(dev(b))
        x, it, nupd, res, status = lat.cg_solve_mixed(mass, 1e-10, 100, z)
        assert (it, nupd, res, status) == (0, 0, 0.0, 0) and not x.any().item()
        x, it, nupd, res, status = lat.cg_solve_mixed(mass, 1e-10, 0, dev(b))
        assert it == 0 and status == 1 and abs(res - 1.0) < 1e-15 and not x.any().item()
        bd = dev(b)
        for bad in (0.0, 1.0, -0.5):
            with pytest.raises(lq.LqcdError):
                lat.cg_solve_mixed(mass, 1e-10, 10, bd, delta=bad)
        with pytest.raises(lq.LqcdError):
            lat.cg_solve_mixed(mass, 1e-10, 10, bd, bd)
        # delta changes the number of updates, not the answer
        xa, ita, na, resa, _ = lat.cg_solve_mixed(mass, 1e-10, 5000, bd, delta=0.5)
        xb, itb, nb, resb, _ = lat.cg_solve_mixed(mass, 1e-10, 5000, bd, delta=0.01)
        assert na > nb >= 1 and resa <= 1e-10 and resb <= 1e-10
        assert rel(xa.cpu().numpy(), xb.cpu().numpy()) <= 1e-8
    uw = synth.gauge_field((4, 4, 4, 4), "smooth", 115)
    with lq.Lattice((4, 4, 4, 4), lq.WILSON) as wl:
        wl.load_gauge(dev(uw))
        with pytest.raises(lq.LqcdError):
            wl.cg_solve_mixed(0.12, 1e-10, 10, dev(synth.source((4, 4, 4, 4), "wilson", 116)))


@pytest.mark.slow
@pytest.mark.parametrize("recon", [18, 12])
def test_mixed_cg_cfg3_bench_workload(lq, recon, cfg3_inputs, cfg3_oracle_cg):
    """32^4 Haar, m = 0.01, in the launch configuration bench.py times: the WHOLE solution against the fp64
    oracle CG of this session (tolerance contract of DESIGN.md 9.3: 1e-8), one oracle application of A,
    and the stored counts of the oracle's mixed solver (make_golden.py --mixed; its solve takes minutes)."""
    c, u, b = cfg3_inputs
    with lattice(lq, c["dims"], u, recon) as lat:
        lat.set_option(lq.OPT_CG_MODE, lq.CG_GRAPH)
        lat.set_option(lq.OPT_CG_CHECK_EVERY, 8)
        x, it, nupd, res, status = lat.cg_solve_mixed(c["param"], c["tol"], 100000, dev(b))
        x = x.cpu().numpy()
    assert status == 0 and res <= c["tol"]
    assert abs(rel(oracle.apply_MdagM(c["dims"], 0, u, c["param"], x), b) - res) <= 1e-3 * res
    assert rel(x, cfg3_oracle_cg["x"]) <= 1e-8
    check_sampled_solution(x, golden("cfg3"), 1e-8)
    m = golden("cfg3_mixed")
    assert count_close(it, m["iters"]) and abs(nupd - m["updates"]) <= 3
