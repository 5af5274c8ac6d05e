"""Parity of the CUDA path (through the C-ABI) with the CPU oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json north_star's: Dslash rel-L2 <= 1e-13 (fp64),
CG solution rel <= 1e-9 at tol 1e-10 with iteration counts within +-2, tables bit-exact."""

import numpy as np
import pytest
import torch

import oracle
from paper_1311_2719_b200 import synth
from lattice_util import check_sampled_solution, golden

pytestmark = pytest.mark.gpu

DSLASH_TOL = 1e-13
CG_TOL = 1e-9

# several tiles of 128 threads plus ragged tails, L = 2 (coincident neighbours), anisotropic shapes
SMALL_SHAPES = [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 8), (6, 4, 2, 2), (2, 6, 4, 10), (10, 6, 6, 4), (8, 8, 8, 8)]


@pytest.fixture(scope="module")
def lq():
    from paper_1311_2719_b200 import lqcd
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return lqcd


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def host(t):
    return t.cpu().numpy()


def fermion_name(f):
    return "staggered" if f == 0 else "wilson"


def make_lattice(lq, dims, fermion, u, recon=18):
    lat = lq.Lattice(dims, fermion)
    lat.set_option(lq.OPT_RECONSTRUCT, recon)
    lat.load_gauge(dev(u))
    return lat


# ------------------------------------------------------------------ tables: bit-exact

@pytest.mark.parametrize("dims", SMALL_SHAPES + [(16, 16, 16, 16), (32, 32, 32, 32), (16, 16, 16, 32)])
def test_tables_bit_exact(lq, dims):
    with lq.Lattice(dims, lq.STAGGERED) as lat:
        iup, idn, l2e = lat.tables()
    o_iup, o_idn, o_l2e = oracle.tables(dims)
    assert np.array_equal(iup.numpy(), o_iup)
    assert np.array_equal(idn.numpy(), o_idn)
    assert np.array_equal(l2e.numpy(), o_l2e)


@pytest.mark.slow
def test_tables_bit_exact_cfg5(lq):
    dims = synth.CONFIGS[5]["dims"]
    with lq.Lattice(dims, lq.STAGGERED) as lat:
        iup, idn, l2e = lat.tables()
    o_iup, o_idn, o_l2e = oracle.tables(dims)
    assert np.array_equal(iup.numpy(), o_iup) and np.array_equal(idn.numpy(), o_idn)
    assert np.array_equal(l2e.numpy(), o_l2e)


# ------------------------------------------------------------------ Dslash and M^+M

@pytest.mark.parametrize("dims", SMALL_SHAPES)
@pytest.mark.parametrize("fermion", [0, 1])
@pytest.mark.parametrize("kind", ["haar", "smooth"])
@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_and_MdagM_small(lq, dims, fermion, kind, recon):
    u = synth.gauge_field(dims, kind, 101)
    shape = oracle._vec_shape(dims, fermion)
    with make_lattice(lq, dims, fermion, u, recon) as lat:
        for parity in (0, 1):
            vin = synth.vector(shape, 102 + parity)
            want = oracle.dslash(dims, fermion, u, parity, vin)
            got = host(lat.dslash(parity, dev(vin)))
            assert rel(got, want) <= DSLASH_TOL
            if fermion == 1:   # the other parity half of the output is left untouched (zero here)
                vh = synth.volume(dims) // 2
                untouched = got[:, :, (1 - parity) * vh:(2 - parity) * vh]
                assert not untouched.any()
        param = 0.07 if fermion == 0 else 0.12
        vin = synth.vector(shape, 104)
        want = oracle.apply_MdagM(dims, fermion, u, param, vin)
        got = host(lat.apply_MdagM(param, dev(vin)))
        assert rel(got, want) <= DSLASH_TOL


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_configs_full_comparison(lq, cfg, recon):
    c, u, b = synth.config_inputs(cfg)
    f = 0 if c["fermion"] == "staggered" else 1
    with make_lattice(lq, c["dims"], f, u, recon) as lat:
        for parity in (0, 1):
            vin = b if f == 1 else synth.vector(b.shape, 200 + parity)
            want = oracle.dslash(c["dims"], f, u, parity, vin)
            got = host(lat.dslash(parity, dev(vin)))
            assert rel(got, want) <= DSLASH_TOL
        want = oracle.apply_MdagM(c["dims"], f, u, c["param"], b)
        got = host(lat.apply_MdagM(c["param"], dev(b)))
        assert rel(got, want) <= DSLASH_TOL


@pytest.mark.slow
def test_dslash_cfg5_sampled_sites_and_norm(lq, cfg5_inputs):
    """48^3 x 96 (6 GB of links): the oracle computes 4096 sampled output sites one by one; the
    rest is covered by anti-hermiticity, <phi, D chi> = -<D phi, chi>, which holds at any size."""
    c, u, b = cfg5_inputs
    dims = c["dims"]
    vh = synth.volume(dims) // 2
    rng = np.random.default_rng(55)
    sites = np.unique(np.concatenate([rng.integers(0, vh, 4000), np.arange(0, 48), np.arange(vh - 48, vh)]))
    with make_lattice(lq, dims, 0, u) as lat:
        chi = synth.vector((3, vh), 501)
        phi = synth.vector((3, vh), 502)
        d_chi = lat.dslash(1, dev(chi))
        d_phi = lat.dslash(0, dev(phi))
        for parity, vin, got in ((1, chi, d_chi), (0, phi, d_phi)):
            want = oracle.dslash_sites(dims, 0, u, parity, vin, sites)
            g = host(got)[:, sites].T
            assert rel(g, want) <= DSLASH_TOL
        lhs = np.vdot(phi.ravel(), host(d_chi).ravel())
        rhs = -np.vdot(host(d_phi).ravel(), chi.ravel())
        assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


# ------------------------------------------------------------------ CG

def run_cg(lat, c, b, mode=None, maxiter=20000, tol=None):
    from paper_1311_2719_b200 import lqcd
    if mode is not None:
        lat.set_option(lqcd.OPT_CG_MODE, mode)
    x, it, res, status = lat.cg_solve(c["param"], c["tol"] if tol is None else tol, maxiter, dev(b))
    return host(x), it, res, status


@pytest.mark.parametrize("cfg", [1, 2, 4])
@pytest.mark.parametrize("recon", [18, 12])
def test_cg_matches_oracle(lq, cfg, recon):
    c, u, b = synth.config_inputs(cfg)
    f = 0 if c["fermion"] == "staggered" else 1
    want = oracle.cg(c["dims"], f, u, c["param"], c["tol"], 20000, b, history=True)
    assert want["status"] == 0
    with make_lattice(lq, c["dims"], f, u, recon) as lat:
        x, it, res, status = run_cg(lat, c, b)
        hist = lat.cg_history().numpy()
    assert status == 0
    assert abs(it - want["iters"]) <= 2
    assert rel(x, want["x"]) <= CG_TOL
    assert res <= 2 * c["tol"] and abs(res - want["true_residual"]) <= 1e-3 * c["tol"] + 0.5 * want["true_residual"]
    # the residual history follows the oracle's while rounding has not yet separated them
    n = min(len(hist), len(want["rr_history"]), 20)
    assert np.allclose(hist[:n], want["rr_history"][:n], rtol=1e-9)


def test_cg_modes_give_identical_iterates(lq):
    c, u, b = synth.config_inputs(1)
    with make_lattice(lq, c["dims"], 0, u) as lat:
        lat.set_option(lq.OPT_PERSISTENT, 0)      # the three-kernel solver and its host loops (auto would pick the one-kernel loop)
        x0, it0, res0, _ = run_cg(lat, c, b, mode=lq.CG_SYNC)
        h0 = lat.cg_history().numpy()
        for every in (1, 3, 16):
            lat.set_option(lq.OPT_CG_CHECK_EVERY, every)
            x1, it1, res1, _ = run_cg(lat, c, b, mode=lq.CG_ASYNC)
            assert it1 == it0 and res1 == res0 and np.array_equal(x0, x1)
            assert np.array_equal(h0, lat.cg_history().numpy())
        x2, it2, res2, _ = run_cg(lat, c, b, mode=lq.CG_GRAPH)
        assert it2 == it0 and res2 == res0 and np.array_equal(x0, x2)


@pytest.mark.parametrize("dims,recon,every", [((4, 4, 4, 4), 18, 8), ((16, 16, 16, 16), 18, 8), ((16, 16, 16, 16), 12, 3),
                                              ((10, 6, 6, 4), 18, 8), ((6, 4, 2, 2), 12, 1), ((2, 2, 2, 2), 18, 8),
                                              ((24, 24, 24, 16), 18, 8)])
def test_cg_persistent_kernel_changes_no_bit(lq, dims, recon, every):
    """The iteration loop as one cooperative kernel (LQCD_OPT_PERSISTENT, cg_persistent.cuh) against the
    three-kernel solver: same arithmetic, same summation order, so solution, iteration count, residual
    history and true residual are bit-identical -- in one physical block (2^4, 4^4: no grid barrier), on
    ragged tiles, with more virtual blocks than resident warps (24^3 x 16: 3456 on 148 x 8), both link
    storages; and both agree with the oracle."""
    mass = 0.05
    u = synth.gauge_field(dims, "haar", 31)
    b = synth.source(dims, "staggered", 32)
    got = {}
    with make_lattice(lq, dims, 0, u, recon) as lat:
        lat.set_option(lq.OPT_CG_MODE, lq.CG_GRAPH)
        lat.set_option(lq.OPT_CG_CHECK_EVERY, every)
        lat.set_option(lq.OPT_STAG_BLOCK, 32)         # a warp of the one-kernel loop = one 32-thread block of the three-kernel path
        for pers in (0, 1):
            lat.set_option(lq.OPT_PERSISTENT, pers)
            n0 = lat.kernel_launches()
            x, it, res, status = lat.cg_solve(mass, 1e-10, 20000, dev(b))
            got[pers] = (host(x), it, res, status, lat.cg_history().numpy(), lat.kernel_launches() - n0)
            xk, itk, _, stk = lat.cg_solve(mass, 0.0, 7, dev(b))                   # tol = 0: exactly 7 iterations
            got[pers] += (host(xk), itk, stk)
    a, p = got[0], got[1]
    assert p[5] == 4 and a[5] > 3 * a[1]              # init + ONE loop kernel + the two kernels of the final check
    assert a[1] == p[1] and a[2] == p[2] and a[3] == p[3] == 0
    assert np.array_equal(a[0], p[0]) and np.array_equal(a[4], p[4])
    assert a[7] == p[7] == 7 and a[8] == p[8] == 1 and np.array_equal(a[6], p[6])
    want = oracle.cg(dims, 0, u, mass, 1e-10, 20000, b)
    assert abs(p[1] - want["iters"]) <= 2 and rel(p[0], want["x"]) <= CG_TOL


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (10, 6, 6, 4)])
def test_cg_persistent_kernel_in_several_launches_changes_no_bit(lq, dims):
    """LQCD_OPT_PERSISTENT_CHUNK: the one-kernel loop cut into launches of 7 iterations (what a solve longer than
    2^20 iterations does, so that the 32-bit arrival counter of the grid barrier cannot wrap) continues from the
    scalars the previous launch left on the device: same iterates, count, history and residual as ONE launch,
    and the number of launches is what the chunking says."""
    mass = 0.05
    u = synth.gauge_field(dims, "haar", 33)
    b = synth.source(dims, "staggered", 34)
    got = {}
    with make_lattice(lq, dims, 0, u) as lat:
        lat.set_option(lq.OPT_PERSISTENT, 1)
        for chunk in (1 << 20, 7):
            lat.set_option(lq.OPT_PERSISTENT_CHUNK, chunk)
            n0 = lat.kernel_launches()
            x, it, res, status = lat.cg_solve(mass, 1e-10, 20000, dev(b))
            assert lat.last_cg_path() == lq.PATH_PERSISTENT
            got[chunk] = (host(x), it, res, status, lat.cg_history().numpy(), lat.kernel_launches() - n0)
            xk, itk, _, stk = lat.cg_solve(mass, 0.0, 15, dev(b))      # tol = 0: exactly 15 = 7 + 7 + 1 iterations
            got[chunk] += (host(xk), itk, stk)
        with pytest.raises(lq.LqcdError):
            lat.set_option(lq.OPT_PERSISTENT_CHUNK, 0)
    one, cut = got[1 << 20], got[7]
    assert one[3] == cut[3] == 0 and one[1] == cut[1] and one[2] == cut[2]
    assert np.array_equal(one[0], cut[0]) and np.array_equal(one[4], cut[4])
    assert one[5] == 4 and cut[5] == 3 + (cut[1] + 6) // 7        # init + loop launches + the two kernels of the final check
    assert one[7] == cut[7] == 15 and one[8] == cut[8] == 1 and np.array_equal(one[6], cut[6])


def test_automatic_one_kernel_loop_respects_an_explicit_host_side_exit_test(lq):
    """On a lattice whose links fit the L2 the default (LQCD_OPT_PERSISTENT = -1) picks the one-kernel loop -- but not
    over a caller who set LQCD_CG_SYNC, the paper's loop with the exit test on the host;
    lqcd_last_cg_path says which loop ran.  The iterates are the same bits either way."""
    dims, mass = (4, 4, 4, 4), 0.1
    u = synth.gauge_field(dims, "haar", 35)
    b = synth.source(dims, "staggered", 36)
    with make_lattice(lq, dims, 0, u) as lat:
        assert lat.last_cg_path() == lq.PATH_NONE
        x0, it0, res0, st0 = lat.cg_solve(mass, 1e-10, 5000, dev(b))
        assert lat.last_cg_path() == lq.PATH_PERSISTENT                      # automatic, nothing set
        lat.set_option(lq.OPT_CG_MODE, lq.CG_GRAPH)
        lat.cg_solve(mass, 1e-10, 5000, dev(b))
        assert lat.last_cg_path() == lq.PATH_PERSISTENT                      # GRAPH / ASYNC leave the choice automatic
        lat.set_option(lq.OPT_CG_MODE, lq.CG_SYNC)
        n0 = lat.kernel_launches()
        x1, it1, res1, st1 = lat.cg_solve(mass, 1e-10, 5000, dev(b))
        assert lat.last_cg_path() == lq.PATH_HOST_LOOP and lat.kernel_launches() - n0 >= 3 * it1
        assert (it0, res0, st0) == (it1, res1, st1) and torch.equal(x0, x1)
        lat.set_option(lq.OPT_PERSISTENT, 1)                                 # an explicit 1 still wins
        lat.cg_solve(mass, 1e-10, 5000, dev(b))
        assert lat.last_cg_path() == lq.PATH_PERSISTENT
        lat.cg_solve_mixed(mass, 1e-10, 5000, dev(b))
        assert lat.last_cg_path() == lq.PATH_HOST_LOOP


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 2), (8, 8, 8, 4)])
def test_wilson_cg_modes_and_the_x_update_in_the_vector_kernel(lq, dims):
    """The Wilson CG does x += alpha p in the vector kernel that follows the update of r (cg_xpupdate_kernel).  The
    three host loops must give the same bits -- the synchronous one launches that kernel once more after the exit
    rule has fired -- and an exit by maxiter must not lose the last update: x_k against the oracle's x_k."""
    kappa = 0.12
    u = synth.gauge_field(dims, "smooth", 41)
    b = synth.source(dims, "wilson", 42)
    want = oracle.cg(dims, 1, u, kappa, 1e-10, 20000, b)
    with make_lattice(lq, dims, 1, u) as lat:
        got = []
        for mode, every in ((lq.CG_SYNC, 1), (lq.CG_ASYNC, 1), (lq.CG_ASYNC, 5), (lq.CG_GRAPH, 8)):
            lat.set_option(lq.OPT_CG_MODE, mode)
            lat.set_option(lq.OPT_CG_CHECK_EVERY, every)
            x, it, res, status = lat.cg_solve(kappa, 1e-10, 20000, dev(b))
            got.append((host(x), it, res, status, lat.cg_history().numpy()))
            for k in (1, 6):
                xk, itk, _, stk = lat.cg_solve(kappa, 0.0, k, dev(b))
                wk = oracle.cg(dims, 1, u, kappa, 0.0, k, b)
                assert itk == k and stk == 1 and rel(host(xk), wk["x"]) <= 1e-12
            xz, itz, resz, stz = lat.cg_solve(kappa, 1e-10, 100, dev(np.zeros_like(b)))
            assert itz == 0 and resz == 0.0 and stz == 0 and not host(xz).any()
    x, it, res, status, h = got[0]
    assert status == 0 and abs(it - want["iters"]) <= 2 and rel(x, want["x"]) <= CG_TOL
    for o in got[1:]:
        assert np.array_equal(o[0], x) and o[1:4] == (it, res, status) and np.array_equal(o[4], h)


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_cg_fixed_iteration_count_matches_oracle_iterate(lq, mode):
    """tol = 0 runs exactly maxiter iterations: compare the iterate x_k itself."""
    c, u, b = synth.config_inputs(2)
    for k in (1, 5, 17):
        want = oracle.cg(c["dims"], 0, u, c["param"], 0.0, k, b)
        with make_lattice(lq, c["dims"], 0, u) as lat:
            lat.set_option(lq.OPT_PERSISTENT, 0)
            x, it, res, status = run_cg(lat, c, b, mode=mode, maxiter=k, tol=0.0)
        assert status == 1 and it == k == want["iters"]
        assert rel(x, want["x"]) <= 1e-12
        assert abs(res - want["true_residual"]) <= 1e-9 * want["true_residual"]


def test_cg_edge_cases(lq):
    c, u, b = synth.config_inputs(1)
    with make_lattice(lq, c["dims"], 0, u) as lat:
        for mode, pers in ((lq.CG_SYNC, 0), (lq.CG_ASYNC, 0), (lq.CG_GRAPH, 0), (lq.CG_GRAPH, 1)):
            lat.set_option(lq.OPT_PERSISTENT, pers)
            x, it, res, status = run_cg(lat, c, np.zeros_like(b), mode=mode)
            assert it == 0 and res == 0.0 and status == 0 and not x.any()          # b = 0
            x, it, res, status = run_cg(lat, c, b, mode=mode, maxiter=0)
            assert it == 0 and status == 1 and not x.any() and abs(res - 1.0) < 1e-15   # no iteration: r = b
            x, it, res, status = run_cg(lat, c, b, mode=mode, maxiter=7)
            assert it == 7 and status == 1
        bd = dev(b)
        with pytest.raises(lq.LqcdError):
            lat.cg_solve(0.1, 1e-10, 10, bd, bd)                                   # aliasing
        with pytest.raises(lq.LqcdError):
            lat.cg_solve(0.1, -1.0, 10, bd)
        with pytest.raises(lq.LqcdError):
            lat.dslash(2, bd)                                                      # bad parity
    with lq.Lattice(c["dims"], 0) as lat2:
        with pytest.raises(lq.LqcdError) as e:
            lat2.dslash(0, dev(b))                                                 # gauge not loaded
        assert e.value.code == -3


def test_host_buffer_entry_points(lq):
    c, u, b = synth.config_inputs(1)
    uh = torch.from_numpy(u).pin_memory()
    bh = torch.from_numpy(b).pin_memory()
    with lq.Lattice(c["dims"], 0) as lat:
        xh, it, res, status = lat.congrad_host(uh, c["param"], c["tol"], 20000, bh)
        x, it2, res2, _ = run_cg(lat, c, b)
        assert status == 0 and it == it2 and res == res2 and np.array_equal(xh.numpy(), x)
        vin = synth.vector(b.shape, 7)
        out = lat.dslash_host(1, torch.from_numpy(vin).pin_memory())
        assert rel(out.numpy(), oracle.dslash(c["dims"], 0, u, 1, vin)) <= DSLASH_TOL


def test_results_are_reproducible_run_to_run(lq):
    c, u, b = synth.config_inputs(2)
    with make_lattice(lq, c["dims"], 0, u) as lat:
        a = run_cg(lat, c, b)
        bres = run_cg(lat, c, b)
    assert a[1] == bres[1] and a[2] == bres[2] and np.array_equal(a[0], bres[0])


# ------------------------------------------------------------------ full-size configs

def _check_against_golden(c, x, it, res, ref):
    assert abs(it - ref["iters"]) <= 2
    check_sampled_solution(x, ref, CG_TOL)
    assert res <= c["tol"] * (1 + 1e-6)      # the true residual itself meets the tolerance (not only the recursion's)


def test_reconstruct_option_invalidates_loaded_gauge(lq):
    c, u, b = synth.config_inputs(1)
    with make_lattice(lq, c["dims"], 0, u) as lat:
        lat.set_option(lq.OPT_RECONSTRUCT, 18)        # unchanged: still loaded
        lat.dslash(1, dev(b))
        lat.set_option(lq.OPT_RECONSTRUCT, 12)
        with pytest.raises(lq.LqcdError) as e:
            lat.dslash(1, dev(b))
        assert e.value.code == -3
        with pytest.raises(lq.LqcdError):
            lat.set_option(lq.OPT_RECONSTRUCT, 8)
        lat.load_gauge(dev(u))
        assert rel(host(lat.dslash(1, dev(b))), oracle.dslash(c["dims"], 0, u, 1, b)) <= DSLASH_TOL


@pytest.mark.slow
@pytest.mark.parametrize("recon", [18, 12])
def test_cg_cfg3_bench_workload(lq, recon, cfg3_inputs, cfg3_oracle_cg):
    """32^4, m = 0.01 in the launch configuration bench.py times, against the oracle's own CG on the same
    inputs: the WHOLE solution vector at rel-L2 <= 1e-9, the iteration count within +-2,
    and the stored oracle reference (tests/golden) which must agree with the oracle run of this session."""
    c, u, b = cfg3_inputs
    with make_lattice(lq, c["dims"], 0, u, recon) as lat:
        lat.set_option(lq.OPT_CG_MODE, lq.CG_GRAPH)
        lat.set_option(lq.OPT_CG_CHECK_EVERY, 8)
        x, it, res, status = lat.cg_solve(c["param"], c["tol"], 50000, dev(b))
        x = host(x)
    want = cfg3_oracle_cg
    assert status == 0 and want["status"] == 0
    assert abs(it - want["iters"]) <= 2
    assert rel(x, want["x"]) <= CG_TOL
    assert abs(res - want["true_residual"]) <= 0.05 * want["true_residual"]
    ax = oracle.apply_MdagM(c["dims"], 0, u, c["param"], x)
    assert abs(rel(ax, b) - res) <= 1e-3 * res + 1e-13
    ref = golden("cfg3")
    assert want["iters"] == ref["iters"]
    check_sampled_solution(want["x"], ref, 1e-12)      # the stored sample is this oracle's solution
    _check_against_golden(c, x, it, res, ref)


@pytest.mark.slow
def test_cg_cfg5(lq, cfg5_inputs):
    """48^3 x 96, m = 0.005 (6 GB of links): iteration count (+-2) and 4096 sampled entries of the oracle's
    solution from tests/golden (the oracle needs ten minutes for this solve), the true residual, and one
    oracle application of A to the whole solution."""
    c, u, b = cfg5_inputs
    with make_lattice(lq, c["dims"], 0, u) as lat:
        x, it, res, status = run_cg(lat, c, b, maxiter=50000)
    assert status == 0
    ax = oracle.apply_MdagM(c["dims"], 0, u, c["param"], x)
    assert abs(rel(ax, b) - res) <= 1e-3 * res + 1e-13
    _check_against_golden(c, x, it, res, golden("cfg5"))
