"""Time-slab decomposition against the oracle of the GLOBAL lattice.

The R slabs of a lattice are driven on the one GPU of the test box through the *_group calls of
include/lqcd_slab.h: the kernels, the peer stores into the neighbours' ghost faces, the slot / flag
mailboxes and the rank-ordered sums are those of an R-GPU run; all slabs share one stream, so no
kernel ever waits for another (B200_PROFILING.md).  The decomposition must not change the
mathematics: the assembled result is compared with the oracle on the undivided lattice at the
north-star tolerances (Dslash 1e-13, CG 1e-9 and +-2 iterations)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1311_2719_b200 import synth
from lattice_util import check_sampled_solution, golden

pytestmark = pytest.mark.gpu

DSLASH_TOL = 1e-13
CG_TOL = 1e-9


@pytest.fixture(scope="module")
def sl():
    from paper_1311_2719_b200 import slab
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return slab


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def group_for(sl, dims, nranks, u, recon=18):
    g = sl.SlabGroup(dims, nranks, recon=recon)
    g.load_gauge_from_global(torch.from_numpy(u))
    return g


def gathered(sl, parts):
    return sl.gather_vector([p.cpu() for p in parts]).numpy()


# lattice, number of slabs: T = 2 (every site on a slab boundary), ragged tiles, the 1-slab ring
# (the periodic wrap itself goes through the mailbox), 16^4 in 2, 4, 8 slabs
CASES = [((4, 4, 4, 4), 1), ((4, 4, 4, 4), 2), ((2, 2, 2, 4), 2), ((4, 2, 6, 8), 4), ((6, 4, 2, 12), 3),
         ((10, 6, 6, 4), 2), ((8, 8, 8, 8), 2), ((8, 8, 8, 8), 4), ((16, 16, 16, 16), 2), ((16, 16, 16, 16), 8)]


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dims,nranks", CASES)
def test_slab_dslash_matches_global_oracle(sl, dims, nranks, recon):
    seed = 4200 + sum(dims) + nranks
    u = synth.gauge_field(dims, "haar", seed)
    vh = synth.volume(dims) // 2
    g = group_for(sl, dims, nranks, u, recon)
    try:
        for parity in (0, 1):
            vin = synth.vector((3, vh), seed + 1 + parity)
            want = oracle.dslash(dims, 0, u, parity, vin)
            outs = g.dslash(parity, g.scatter(torch.from_numpy(vin)), g.new_vectors())
            g.synchronize()
            assert rel(gathered(sl, outs), want) <= DSLASH_TOL
        # twice in a row with different inputs: the two ghost buffers alternate
        for k in range(3):
            vin = synth.vector((3, vh), seed + 10 + k)
            outs = g.dslash(1, g.scatter(torch.from_numpy(vin)), g.new_vectors())
            g.synchronize()
            assert rel(gathered(sl, outs), oracle.dslash(dims, 0, u, 1, vin)) <= DSLASH_TOL
    finally:
        g.close()


@pytest.mark.parametrize("dims,nranks", [((4, 4, 4, 4), 2), ((4, 2, 6, 8), 4), ((8, 8, 8, 8), 2), ((16, 16, 16, 16), 4)])
def test_slab_MdagM_matches_global_oracle(sl, dims, nranks):
    u = synth.gauge_field(dims, "smooth", 77 + nranks)
    vin = synth.vector((3, synth.volume(dims) // 2), 78)
    want = oracle.apply_MdagM(dims, 0, u, 0.07, vin)
    g = group_for(sl, dims, nranks, u)
    try:
        outs = g.apply_MdagM(0.07, g.scatter(torch.from_numpy(vin)), g.new_vectors())
        g.synchronize()
        assert rel(gathered(sl, outs), want) <= DSLASH_TOL
    finally:
        g.close()


def test_slab_boundary_sign_sits_on_the_global_boundary(sl):
    """Unit links, constant vector: D v vanishes except on the two time-slices next to the GLOBAL
    antiperiodic boundary, wherever the slabs are cut (reading A4)."""
    dims, nranks = (4, 4, 4, 8), 4
    v, vh, sh = synth.volume(dims), synth.volume(dims) // 2, 4 * 4 * 4 // 2
    u = np.zeros((v, 4, 3, 3), complex)
    u[:, :, [0, 1, 2], [0, 1, 2]] = 1.0
    vin = np.ones((3, vh), complex)
    g = group_for(sl, dims, nranks, u)
    try:
        outs = g.dslash(1, g.scatter(torch.from_numpy(vin)), g.new_vectors())
        g.synchronize()
        out = gathered(sl, outs).reshape(3, 8, sh)
        assert np.abs(out[:, 1:7]).max() == 0.0
        assert np.abs(np.abs(out[:, 0]) - 1.0).max() < 1e-15 and np.abs(np.abs(out[:, 7]) - 1.0).max() < 1e-15
        assert rel(out.reshape(3, vh), oracle.dslash(dims, 0, u, 1, vin)) <= DSLASH_TOL
    finally:
        g.close()


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("cfg,nranks", [(1, 1), (1, 2), (2, 2), (2, 4), (2, 8)])
def test_slab_cg_matches_global_oracle(sl, cfg, nranks, recon):
    c, u, b = synth.config_inputs(cfg)
    want = oracle.cg(c["dims"], 0, u, c["param"], c["tol"], 20000, b)
    assert want["status"] == 0
    g = group_for(sl, c["dims"], nranks, u, recon)
    try:
        xs, it, res, status = g.cg_solve(c["param"], c["tol"], 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        x = gathered(sl, xs)
        assert status == 0
        assert abs(it - want["iters"]) <= 2
        assert rel(x, want["x"]) <= CG_TOL
        assert res <= 2 * c["tol"]
        # three synchronisation points per iteration, in step on every rank
        assert len({s.sync_points() for s in g.slabs}) == 1
    finally:
        g.close()


def test_slab_cg_fixed_iterations_and_rank_count_independence(sl):
    """tol = 0: exactly k iterations.  The iterate agrees with the oracle's to rounding for every
    number of slabs, and the batch size of the host loop does not change a bit of it."""
    c, u, b = synth.config_inputs(2)
    for k in (1, 6):
        want = oracle.cg(c["dims"], 0, u, c["param"], 0.0, k, b)
        for nranks in (1, 2, 8):
            g = group_for(sl, c["dims"], nranks, u)
            try:
                ref = None
                for every in (1, 5):
                    g.set_option(sl.OPT_CHECK_EVERY, every)
                    xs, it, res, status = g.cg_solve(c["param"], 0.0, k, g.scatter(torch.from_numpy(b)), g.new_vectors())
                    x = gathered(sl, xs)
                    assert status == 1 and it == k
                    assert rel(x, want["x"]) <= 1e-12
                    assert abs(res - want["true_residual"]) <= 1e-9 * want["true_residual"]
                    if ref is None:
                        ref = x
                    assert np.array_equal(ref, x)
            finally:
                g.close()


@pytest.mark.parametrize("nranks", [1, 4])
def test_slab_cg_graph_replay_changes_no_bit(sl, nranks):
    """LQCD_SLAB_OPT_GRAPH: the batch of iterations replayed from a CUDA graph (synchronisation numbers
    counted on the device, ghost buffers alternating inside the graph) against kernel-by-kernel launches."""
    c, u, b = synth.config_inputs(2)
    g = group_for(sl, c["dims"], nranks, u)
    try:
        got = []
        for graph, every in ((0, 4), (1, 4), (1, 3), (1, 16)):
            g.set_option(sl.OPT_GRAPH, graph)
            g.set_option(sl.OPT_CHECK_EVERY, every)
            xs, it, res, status = g.cg_solve(c["param"], c["tol"], 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
            got.append((gathered(sl, xs), it, res, status))
        for x, it, res, status in got[1:]:
            assert status == 0 and it == got[0][1] and res == got[0][2] and np.array_equal(x, got[0][0])
        assert len({s.sync_points() for s in g.slabs}) == 1
    finally:
        g.close()


def test_slab_cg_agrees_with_the_single_gpu_solver(sl):
    from paper_1311_2719_b200 import lqcd
    c, u, b = synth.config_inputs(2)
    with lqcd.Lattice(c["dims"], lqcd.STAGGERED) as lat:
        lat.load_gauge(torch.from_numpy(u).cuda())
        x1, it1, res1, st1 = lat.cg_solve(c["param"], c["tol"], 20000, torch.from_numpy(b).cuda())
        x1 = x1.cpu().numpy()
    g = group_for(sl, c["dims"], 4, u)
    try:
        xs, it, res, status = g.cg_solve(c["param"], c["tol"], 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        assert status == st1 == 0 and abs(it - it1) <= 2
        assert rel(gathered(sl, xs), x1) <= CG_TOL
    finally:
        g.close()


def test_slab_single_rank_entry_points(sl):
    """lqcd_slab_dslash / _apply_MdagM / _cg_solve: the one-rank-per-process calls, here on the 1-slab
    ring (its own neighbour on both sides), where signal and wait follow each other on one stream."""
    c, u, b = synth.config_inputs(1)
    dims = c["dims"]
    s = sl.Slab(dims, 0, 1)
    try:
        s.connect([s.mailbox_ptr])
        ug = torch.from_numpy(u)
        s.load_gauge(sl.local_gauge(ug, dims, 0, 1).cuda(), sl.u3_below_from_global(ug, dims, 0, 1).cuda())
        vin = synth.vector((3, synth.volume(dims) // 2), 5)
        out = s.dslash(1, torch.from_numpy(vin).cuda(), s.new_vector())
        s.stream.synchronize()
        assert rel(out.cpu().numpy(), oracle.dslash(dims, 0, u, 1, vin)) <= DSLASH_TOL
        out = s.apply_MdagM(0.1, torch.from_numpy(vin).cuda(), s.new_vector())
        s.stream.synchronize()
        assert rel(out.cpu().numpy(), oracle.apply_MdagM(dims, 0, u, 0.1, vin)) <= DSLASH_TOL
        want = oracle.cg(dims, 0, u, c["param"], c["tol"], 20000, b)
        x, it, res, status = s.cg_solve(c["param"], c["tol"], 20000, torch.from_numpy(b).cuda(), s.new_vector())
        assert status == 0 and abs(it - want["iters"]) <= 2 and rel(x.cpu().numpy(), want["x"]) <= CG_TOL
    finally:
        s.close()


def test_slab_fused_synchronisation_changes_no_bit(sl):
    """One rank per process: the synchronisation point inside the last block of the producer kernels
    (LQCD_SLAB_OPT_FUSE_SYNC, default) against separate launches, with and without graph replay, and
    against the group call on the same 1-slab ring."""
    c, u, b = synth.config_inputs(2)
    dims = c["dims"]
    ug = torch.from_numpy(u)
    s = sl.Slab(dims, 0, 1)
    g = group_for(sl, dims, 1, u)
    try:
        s.connect([s.mailbox_ptr])
        s.load_gauge(sl.local_gauge(ug, dims, 0, 1).cuda(), sl.u3_below_from_global(ug, dims, 0, 1).cuda())
        got = []
        for fuse, graph in ((1, 1), (1, 0), (0, 1), (0, 0)):
            s.set_option(sl.OPT_FUSE_SYNC, fuse)
            s.set_option(sl.OPT_GRAPH, graph)
            before = s.kernel_launches()
            x, it, res, status = s.cg_solve(c["param"], c["tol"], 20000, torch.from_numpy(b).cuda(), s.new_vector())
            got.append((x.cpu().numpy(), it, res, status, s.kernel_launches() - before))
        xs, it, res, status = g.cg_solve(c["param"], c["tol"], 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        got.append((gathered(sl, xs), it, res, status, 0))
        for x, it, res, status, _ in got[1:]:
            assert status == 0 and it == got[0][1] and res == got[0][2] and np.array_equal(x, got[0][0])
        assert got[0][4] < got[2][4]            # fused: three launches per iteration instead of six
        want = oracle.cg(dims, 0, u, c["param"], c["tol"], 20000, b)
        assert abs(got[0][1] - want["iters"]) <= 2 and rel(got[0][0], want["x"]) <= CG_TOL
    finally:
        s.close()
        g.close()


def test_slab_system_scope_release_acquire_changes_no_bit(sl):
    """LQCD_SLAB_OPT_ACQUIRE = 1 (the fences a peer on another GPU gets by default) forced on one GPU: the ring of one
    rank with the fused tail and with separate launches, same bits as without; automatic = off here (the
    mailbox is on the same device), and the option rejects other values."""
    c, u, b = synth.config_inputs(1)
    dims = c["dims"]
    ug = torch.from_numpy(u)
    s = sl.Slab(dims, 0, 1)
    try:
        s.connect([s.mailbox_ptr])
        s.load_gauge(sl.local_gauge(ug, dims, 0, 1).cuda(), sl.u3_below_from_global(ug, dims, 0, 1).cuda())
        got = []
        for acquire, fuse in ((-1, 1), (1, 1), (1, 0), (0, 0)):
            s.set_option(sl.OPT_ACQUIRE, acquire)
            s.set_option(sl.OPT_FUSE_SYNC, fuse)
            x, it, res, status = s.cg_solve(c["param"], c["tol"], 20000, torch.from_numpy(b).cuda(), s.new_vector())
            got.append((x.cpu().numpy(), it, res, status))
        for x, it, res, status in got[1:]:
            assert status == 0 and it == got[0][1] and res == got[0][2] and np.array_equal(x, got[0][0])
        want = oracle.cg(dims, 0, u, c["param"], c["tol"], 20000, b)
        assert abs(got[0][1] - want["iters"]) <= 2 and rel(got[0][0], want["x"]) <= CG_TOL
        with pytest.raises(Exception):
            s.set_option(sl.OPT_ACQUIRE, 2)
    finally:
        s.close()


def test_slab_edge_cases_and_errors(sl):
    c, u, b = synth.config_inputs(1)
    dims = c["dims"]
    g = group_for(sl, dims, 2, u)
    try:
        zero = [torch.zeros_like(v) for v in g.scatter(torch.from_numpy(b))]
        xs, it, res, status = g.cg_solve(0.1, 1e-10, 100, zero, g.new_vectors())          # b = 0 (reading A11)
        assert it == 0 and res == 0.0 and status == 0 and not gathered(sl, xs).any()
        xs, it, res, status = g.cg_solve(0.1, 1e-10, 0, g.scatter(torch.from_numpy(b)), g.new_vectors())
        assert it == 0 and status == 1 and abs(res - 1.0) < 1e-15                          # no iteration: r = b
        bs = g.scatter(torch.from_numpy(b))
        with pytest.raises(sl.LqcdError):
            g.cg_solve(0.1, 1e-10, 10, bs, bs)                                             # aliasing
        with pytest.raises(sl.LqcdError):
            g.dslash(2, bs, g.new_vectors())                                               # bad parity
    finally:
        g.close()
    with pytest.raises(ValueError):
        sl.SlabGroup((4, 4, 4, 4), 4)                                                      # T = 1
    with pytest.raises(ValueError):
        sl.SlabGroup((4, 4, 4, 6), 4)                                                      # 6 % 4
    with pytest.raises(sl.LqcdError):
        sl.Slab((4, 4, 4, 12), 0, 4)                                                       # T = 3 is odd
    s = sl.Slab(dims, 0, 2)
    try:
        with pytest.raises(sl.LqcdError) as e:                                             # peers not connected
            s.dslash(1, s.new_vector(), s.new_vector())
        assert e.value.code == -3
    finally:
        s.close()


@pytest.mark.slow
@pytest.mark.parametrize("nranks", [1, 4])
def test_slab_cg_cfg3_bench_workload(sl, nranks, cfg3_inputs, cfg3_oracle_cg):
    """32^4, m = 0.01 as `bench.py --parallelism slab` times it (nranks = 1: lqcd_slab_cg_solve with the fused
    synchronisation tail and graph replay) and cut into four slabs, against the oracle's own CG on the
    UNDIVIDED lattice (run once per session): whole assembled solution at 1e-9, iterations +-2, the stored
    sample (tests/golden) and one oracle application of A."""
    c, u, b = cfg3_inputs
    dims = c["dims"]
    if nranks == 1:
        ug = torch.from_numpy(u)
        s = sl.Slab(dims, 0, 1)
        try:
            s.connect([s.mailbox_ptr])
            s.load_gauge(sl.local_gauge(ug, dims, 0, 1).cuda(), sl.u3_below_from_global(ug, dims, 0, 1).cuda())
            xt, it, res, status = s.cg_solve(c["param"], c["tol"], 50000, torch.from_numpy(b).cuda(), s.new_vector())
            x = xt.cpu().numpy()
        finally:
            s.close()
    else:
        g = group_for(sl, dims, nranks, u)
        try:
            xs, it, res, status = g.cg_solve(c["param"], c["tol"], 50000, g.scatter(torch.from_numpy(b)), g.new_vectors())
            x = gathered(sl, xs)
        finally:
            g.close()
    want = cfg3_oracle_cg
    assert status == 0 and res <= c["tol"] * (1 + 1e-6) and abs(it - want["iters"]) <= 2
    assert rel(x, want["x"]) <= CG_TOL
    check_sampled_solution(x, golden("cfg3"), CG_TOL)
    ax = oracle.apply_MdagM(dims, 0, u, c["param"], x)
    assert abs(rel(ax, b) - res) <= 1e-3 * res + 1e-13


@pytest.mark.slow
def test_slab_cg_cfg5_eight_slabs(sl, cfg5_inputs):
    """48^3 x 96 (6 GB of links) cut into eight slabs of 12 time-slices, as an 8-GPU run would hold it: the
    assembled solution against the oracle's stored iteration count and 4096 sampled solution entries
    (tests/golden) and one oracle application of A (holds at any size)."""
    c, u, b = cfg5_inputs
    dims = c["dims"]
    g = group_for(sl, dims, 8, u)
    try:
        xs, it, res, status = g.cg_solve(c["param"], c["tol"], 50000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        x = gathered(sl, xs)
    finally:
        g.close()
    assert status == 0 and res <= c["tol"] * (1 + 1e-6)
    ax = oracle.apply_MdagM(dims, 0, u, c["param"], x)
    assert abs(rel(ax, b) - res) <= 1e-3 * res + 1e-13
    ref = golden("cfg5")
    assert abs(it - ref["iters"]) <= 2
    check_sampled_solution(x, ref, CG_TOL)


# ------------------------------------------------------------------ mixed precision on slabs (SURVEY.md 8(f) rows 3 + 4b)
def _count_close(a, b):
    return abs(a - b) <= max(3, 0.03 * b)


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dims,kind,mass,nranks", [((4, 4, 4, 4), "random_su3", 0.1, 1), ((4, 4, 4, 4), "random_su3", 0.1, 2),
                                                   ((6, 4, 2, 12), "smooth", 0.05, 3), ((8, 8, 8, 8), "haar", 0.03, 2),
                                                   ((8, 8, 8, 8), "haar", 0.03, 4), ((16, 16, 16, 16), "smooth", 0.05, 4),
                                                   ((16, 16, 16, 16), "smooth", 0.05, 8)])
def test_slab_mixed_cg_matches_global_mixed_oracle(sl, dims, kind, mass, nranks, recon):
    """lqcd_slab_cg_solve_mixed_group against the oracle's mixed-precision CG and its fp64 CG on the UNDIVIDED lattice,
    under the contract of tests/test_gpu_mixed.py: exit declared on an fp64 residual (true residual
    <= tol), solution within the bound two tol-converged solutions obey (and 1e-8), iteration / update counts within
    a few per cent / +-2 (fp32 rounding and the grouping of the sums perturb the trajectory), first residuals to
    fp32 accuracy."""
    tol = 1e-10
    u = synth.gauge_field(dims, kind, 111)
    b = synth.source(dims, "staggered", 112)
    want = oracle.cg_mixed(dims, u, mass, tol, 20000, b, history=True)
    plain = oracle.cg(dims, 0, u, mass, tol, 20000, b)
    assert want["status"] == 0
    g = group_for(sl, dims, nranks, u, recon)
    try:
        g.set_option(sl.OPT_CHECK_EVERY, 4)
        xs, it, nupd, res, status = g.cg_solve_mixed(mass, tol, 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        x = gathered(sl, xs)
    finally:
        g.close()
    assert status == 0 and res <= tol
    bound = 2 * tol * np.linalg.norm(b) / mass ** 2
    assert np.linalg.norm(x - plain["x"]) <= min(bound, 1e-8 * np.linalg.norm(plain["x"]))
    assert np.linalg.norm(x - want["x"]) <= min(bound, 1e-8 * np.linalg.norm(want["x"]))
    assert _count_close(it, want["iters"]) and abs(nupd - want["updates"]) <= 2
    true = rel(oracle.apply_MdagM(dims, 0, u, mass, x), b)
    assert abs(true - res) <= 1e-3 * true + 1e-15


def test_slab_mixed_cg_agrees_with_the_single_gpu_mixed_solver_and_batching(sl):
    """The decomposition and the batch size must not change the mixed solver: counts as the undivided solver's, the
    same solution to far below the contract, bit-identical results whatever check_every, edge cases."""
    from paper_1311_2719_b200 import lqcd
    c, u, b = synth.config_inputs(2)
    with lqcd.Lattice(c["dims"], lqcd.STAGGERED) as lat:
        lat.load_gauge(torch.from_numpy(u).cuda())
        x1, it1, n1, res1, st1 = lat.cg_solve_mixed(c["param"], c["tol"], 20000, torch.from_numpy(b).cuda())
        x1 = x1.cpu().numpy()
    g = group_for(sl, c["dims"], 4, u)
    try:
        got = []
        for every in (1, 8):
            g.set_option(sl.OPT_CHECK_EVERY, every)
            xs, it, nupd, res, status = g.cg_solve_mixed(c["param"], c["tol"], 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
            got.append((gathered(sl, xs), it, nupd, res, status))
        assert got[0][1:] == got[1][1:] and np.array_equal(got[0][0], got[1][0])
        x, it, nupd, res, status = got[0]
        assert status == st1 == 0 and _count_close(it, it1) and abs(nupd - n1) <= 2 and res <= c["tol"]
        assert rel(x, x1) <= 1e-8
        # b = 0, maxiter = 0, a fixed number of iterations (tol = 0)
        zero = [torch.zeros_like(v) for v in g.scatter(torch.from_numpy(b))]
        xs, it, nupd, res, status = g.cg_solve_mixed(c["param"], c["tol"], 100, zero, g.new_vectors())
        assert it == 0 and res == 0.0 and status == 0 and not gathered(sl, xs).any()
        xs, it, nupd, res, status = g.cg_solve_mixed(c["param"], c["tol"], 0, g.scatter(torch.from_numpy(b)), g.new_vectors())
        assert it == 0 and status == 1 and not gathered(sl, xs).any()
        xs, it, nupd, res, status = g.cg_solve_mixed(c["param"], 0.0, 9, g.scatter(torch.from_numpy(b)), g.new_vectors())
        assert it == 9 and status == 1
        want = oracle.cg(c["dims"], 0, u, c["param"], 0.0, 9, b)
        assert rel(gathered(sl, xs), want["x"]) <= 2e-5          # nine fp32 iterations against nine fp64 ones
        # and the fp64 slab solver on the same slabs is not disturbed by the mixed one's state
        xs, it, res, status = g.cg_solve(c["param"], c["tol"], 20000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        full = oracle.cg(c["dims"], 0, u, c["param"], c["tol"], 20000, b)
        assert status == 0 and abs(it - full["iters"]) <= 2 and rel(gathered(sl, xs), full["x"]) <= CG_TOL
    finally:
        g.close()


@pytest.mark.slow
@pytest.mark.parametrize("recon", [18, 12])
def test_slab_mixed_cg_cfg3_bench_workload(sl, recon, cfg3_inputs, cfg3_oracle_cg):
    """The bench workload (32^4, m = 0.01) through the mixed-precision slab solver in two slabs, against the oracle's
    fp64 CG on the undivided lattice (run once per session): the contract of DESIGN.md 9.3 -- true residual <= tol,
    the WHOLE solution within 1e-8 -- plus the stored 4096-entry sample and one oracle application of A."""
    c, u, b = cfg3_inputs
    dims = c["dims"]
    g = group_for(sl, dims, 2, u, recon)
    try:
        xs, it, nupd, res, status = g.cg_solve_mixed(c["param"], c["tol"], 50000, g.scatter(torch.from_numpy(b)), g.new_vectors())
        x = gathered(sl, xs)
    finally:
        g.close()
    want = cfg3_oracle_cg
    assert status == 0 and res <= c["tol"] and nupd >= 5
    assert _count_close(it, want["iters"])             # reliable updates cost no convergence (3141 against 3138 undivided)
    assert rel(x, want["x"]) <= 1e-8
    check_sampled_solution(x, golden("cfg3"), 1e-8)
    ax = oracle.apply_MdagM(dims, 0, u, c["param"], x)
    assert abs(rel(ax, b) - res) <= 1e-3 * res + 1e-13


def test_slab_mixed_single_rank_entry_point(sl):
    c, u, b = synth.config_inputs(1)
    dims = c["dims"]
    s = sl.Slab(dims, 0, 1)
    try:
        s.connect([s.mailbox_ptr])
        ug = torch.from_numpy(u)
        s.load_gauge(sl.local_gauge(ug, dims, 0, 1).cuda(), sl.u3_below_from_global(ug, dims, 0, 1).cuda())
        want = oracle.cg(dims, 0, u, c["param"], c["tol"], 20000, b)
        x, it, nupd, res, status = s.cg_solve_mixed(c["param"], c["tol"], 20000, torch.from_numpy(b).cuda(), s.new_vector())
        assert status == 0 and res <= c["tol"] and nupd >= 1 and rel(x.cpu().numpy(), want["x"]) <= 1e-8
    finally:
        s.close()


# ------------------------------------------------------------------ CUDA IPC plumbing, two processes on the one GPU
def _ipc_worker(rank, world, port, out):
    """Maps the peer's mailbox through lqcd_slab_ipc_export / _open and moves bytes with plain copies.
    No compute call is made: kernels of two processes that wait for each other must not share a GPU."""
    import ctypes
    import os
    import sys
    os.environ.update(RANK=str(rank), LOCAL_RANK="0", WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import torch
    import torch.distributed as dist
    from paper_1311_2719_b200 import slab as sl
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ok, msg = False, ""
    try:
        dims = (8, 8, 8, 8)
        s = sl.Slab(dims, rank, world, device="cuda:0")
        s.connect_ipc()                                     # all-gather of the handles over gloo, open, connect, barrier
        lib = s._lib
        # the peer's mailbox as this process sees it: write a pattern at a rank-dependent offset of its ghost area
        nbytes = lib.lqcd_slab_mailbox_bytes(s._s)
        other = 1 - rank
        peer_ptr = s._opened[0][0]
        pattern = torch.full((1024,), 100.0 + rank, dtype=torch.float64, device="cuda:0")
        off = nbytes - 2 * 8192 + rank * 8192              # the tail of the ghost faces: unused by anything else here
        try:
            rt = ctypes.CDLL("libcudart.so.12")            # the runtime torch has already loaded
        except OSError:
            rt = ctypes.CDLL("/usr/local/cuda/lib64/libcudart.so.12")
        rt.cudaMemcpy.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int]
        rc = rt.cudaMemcpy(ctypes.c_void_p(peer_ptr + off), ctypes.c_void_p(pattern.data_ptr()), 8192, 3)
        torch.cuda.synchronize()
        dist.barrier()
        # what the peer wrote into MY mailbox
        mine = torch.empty(1024, dtype=torch.float64, device="cuda:0")
        rc2 = rt.cudaMemcpy(ctypes.c_void_p(mine.data_ptr()), ctypes.c_void_p(s.mailbox_ptr + nbytes - 2 * 8192 + other * 8192), 8192, 3)
        torch.cuda.synchronize()
        ok = rc == 0 and rc2 == 0 and bool((mine == 100.0 + other).all().item())
        dist.barrier()
        s.close()
    except Exception as e:  # pragma: no cover - reported through the queue
        msg = repr(e)
    out.put(dict(rank=rank, ok=ok, msg=msg))
    dist.destroy_process_group()


def test_slab_ipc_mailboxes_between_two_processes():
    import socket
    import torch.multiprocessing as mp
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_ipc_worker, args=(i, 2, port, q)) for i in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=300) for _ in procs), key=lambda d: d["rank"])
    for p in procs:
        p.join(timeout=120)
    assert all(g["ok"] for g in got), got


# ------------------------------------------------------------------ two GPUs, one process each (runs only where two are visible)
def _two_gpu_worker(rank, world, port, fuse, acquire, out):
    """One rank per process and per GPU: IPC-mapped mailboxes, face stores and flags over NVLink, compute calls on
    both sides -- the configuration a one-GPU box cannot run (two kernels that wait on one another must not
    share a GPU).  Each rank reports its slab of D b, A b and the CG solution; the parent compares the
    assembled vectors with the oracle of the undivided lattice."""
    import os
    import sys
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import torch
    import torch.distributed as dist
    from paper_1311_2719_b200 import slab as sl, synth
    res, msg = None, ""
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dims, mass = (8, 8, 8, 8), 0.1
        dev = torch.device("cuda", rank)
        torch.cuda.set_device(dev)
        u = torch.from_numpy(synth.gauge_field(dims, "haar", 7))
        b = torch.from_numpy(synth.source(dims, "staggered", 8))
        s = sl.Slab(dims, rank, world, device=dev)
        s.set_option(sl.OPT_TIMEOUT_MS, 5000)
        s.set_option(sl.OPT_FUSE_SYNC, fuse)
        s.set_option(sl.OPT_ACQUIRE, acquire)
        s.connect_ipc()
        ul = sl.local_gauge(u, dims, rank, world)
        ub = sl.exchange_u3_below(ul, dims, rank, world)      # the set-up exchange over torch.distributed
        s.load_gauge(ul.to(dev), ub.to(dev))
        bl = sl.local_vector(b, dims, rank, world).to(dev)
        d, a, x = s.new_vector(), s.new_vector(), s.new_vector()
        s.dslash(1, bl, d)
        s.apply_MdagM(mass, bl, a)
        _, it, tr, st = s.cg_solve(mass, 1e-10, 5000, bl, x)
        s.stream.synchronize()
        res = dict(d=d.cpu().numpy(), a=a.cpu().numpy(), x=x.cpu().numpy(), iters=it, true_residual=tr, status=st,
                   sync_points=s.sync_points())
        dist.barrier()
        s.close()
    except Exception as e:  # pragma: no cover - reported through the queue
        msg = repr(e)
    out.put(dict(rank=rank, res=res, msg=msg))
    dist.destroy_process_group()


@pytest.mark.parametrize("acquire", [-1, 1, 0])   # -1: automatic (on: the peer is another GPU); 0: relaxed words only
@pytest.mark.parametrize("fuse", [0, 1])
def test_slab_two_gpus_one_process_each(fuse, acquire):
    import socket
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs: kernels of two ranks that wait on one another must not share a device")
    import oracle
    from paper_1311_2719_b200 import synth
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_two_gpu_worker, args=(i, 2, port, fuse, acquire, q)) for i in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=600) for _ in procs), key=lambda g: g["rank"])
    for p in procs:
        p.join(timeout=120)
    assert all(g["res"] is not None for g in got), [g["msg"] for g in got]
    dims, mass = (8, 8, 8, 8), 0.1
    u = synth.gauge_field(dims, "haar", 7)
    b = synth.source(dims, "staggered", 8)
    cat = lambda k: np.concatenate([g["res"][k] for g in got], axis=1)
    assert rel(cat("d"), oracle.dslash(dims, 0, u, 1, b)) <= 1e-13
    assert rel(cat("a"), oracle.apply_MdagM(dims, 0, u, mass, b)) <= 1e-13
    want = oracle.cg(dims, 0, u, mass, 1e-10, 5000, b)
    assert got[0]["res"]["iters"] == got[1]["res"]["iters"] and abs(got[0]["res"]["iters"] - want["iters"]) <= 2
    assert got[0]["res"]["true_residual"] == got[1]["res"]["true_residual"]      # rank-ordered sums: bit-identical scalars
    assert all(g["res"]["status"] == 0 for g in got)
    assert rel(cat("x"), want["x"]) <= 1e-9
