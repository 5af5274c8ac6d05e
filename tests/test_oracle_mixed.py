"""Pins for the oracle's mixed-precision CG with reliable updates (the
technique of the paper's reference [2]).

P11: whatever happens in fp32, the result has a plain definition -- x = A^-1 b to the stated
tolerance -- so the mixed solver is pinned by Gaussian elimination of the dense matrix on 2^4, by the
fp64 residual recomputed here from the (pinned) fp64 operator, and by the plain fp64 CG.  The fp32
hopping term is pinned to the fp64 one within fp32 rounding (and shown to really be fp32).  No GPU.
"""
import numpy as np
import pytest

import oracle
from oracle import STAGGERED
from paper_1311_2719_b200 import synth


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (4, 2, 6, 4)])
@pytest.mark.parametrize("kind", ["haar", "smooth"])
def test_fp32_hopping_term_is_the_fp64_one_within_fp32_rounding(dims, kind):
    u = synth.gauge_field(dims, kind, 101)
    v = synth.source(dims, "staggered", 102)
    for parity in (0, 1):
        d64 = oracle.dslash(dims, STAGGERED, u, parity, v)
        d32 = oracle.stag_dslash_f32(dims, u, parity, v)
        e = rel(d32, d64)
        assert 1e-9 < e < 5e-7, e     # 8 hops x 3 products of fl32 operands: a few units of 6e-8


def test_mixed_cg_against_dense_solve_on_2_4():
    dims, mass = (2, 2, 2, 2), 0.1
    u = synth.gauge_field(dims, "haar", 103)
    b = synth.source(dims, "staggered", 104)
    n = b.size
    a = np.empty((n, n), complex)
    for j in range(n):
        e = np.zeros(n, complex)
        e[j] = 1.0
        a[:, j] = oracle.apply_MdagM(dims, STAGGERED, u, mass, e.reshape(b.shape)).ravel()
    x_dense = np.linalg.solve(a, b.ravel()).reshape(b.shape)
    r = oracle.cg_mixed(dims, u, mass, 1e-12, 2000, b)
    assert r["status"] == 0 and r["updates"] >= 2
    assert rel(r["x"], x_dense) < 1e-9
    assert r["true_residual"] <= 1e-12


@pytest.mark.parametrize("cfg,delta", [(1, 0.1), (1, 0.5), (1, 0.01)])
def test_mixed_cg_reaches_the_fp64_tolerance_and_the_fp64_solution(cfg, delta):
    c, u, b = synth.config_inputs(cfg)
    dims, mass, tol = c["dims"], c["param"], c["tol"]
    want = oracle.cg(dims, STAGGERED, u, mass, tol, 20000, b)
    r = oracle.cg_mixed(dims, u, mass, tol, 20000, b, delta=delta, history=True)
    assert r["status"] == 0
    # the residual from its definition, recomputed here with the fp64 operator
    res = np.linalg.norm(b - oracle.apply_MdagM(dims, STAGGERED, u, mass, r["x"])) / np.linalg.norm(b)
    assert res <= tol and abs(res - r["true_residual"]) <= 1e-6 * res
    # both are within tol of the same solution: |x1 - x2| <= 2 tol |b| / lambda_min, lambda_min >= m^2
    bound = 2 * tol * np.linalg.norm(b) / mass ** 2 / np.linalg.norm(want["x"])
    assert rel(r["x"], want["x"]) <= min(bound, 1e-8)
    # the final exit is itself an update; a residual can fall by more than delta in one step, so the
    # count has no sharper lower bound, but it cannot exceed one per factor delta plus the rises
    assert 1 <= r["updates"] <= r["iters"]
    # fp32 costs a few iterations, not many
    assert want["iters"] <= r["iters"] + 2 and r["iters"] <= 1.25 * want["iters"] + 10
    # the history's last entry is the fp64 residual the exit was declared on
    assert np.isclose(np.sqrt(r["rr_history"][-1]) / np.linalg.norm(b), r["true_residual"], rtol=1e-9)


def test_mixed_cg_edge_cases():
    dims = (4, 4, 4, 4)
    u = synth.gauge_field(dims, "haar", 105)
    b = synth.source(dims, "staggered", 106)
    z = np.zeros_like(b)
    r = oracle.cg_mixed(dims, u, 0.1, 1e-10, 100, z)
    assert r["status"] == 0 and r["iters"] == 0 and r["updates"] == 0 and r["true_residual"] == 0 and not r["x"].any()
    r = oracle.cg_mixed(dims, u, 0.1, 1e-10, 5, b)
    assert r["status"] == 1 and r["iters"] == 5
    # the partial solution is returned: its residual is what 5 CG iterations reach (below |b|)
    res = np.linalg.norm(b - oracle.apply_MdagM(dims, STAGGERED, u, 0.1, r["x"])) / np.linalg.norm(b)
    assert abs(res - r["true_residual"]) <= 1e-9 * res and res < 1.0
    want = oracle.cg(dims, STAGGERED, u, 0.1, 0.0, 5, b)
    assert rel(r["x"], want["x"]) < 1e-5           # the first iterates are the fp64 ones to fp32 rounding
    r0 = oracle.cg_mixed(dims, u, 0.1, 0.0, 40, b)  # tol = 0: exactly maxiter iterations, updates by delta only
    assert r0["status"] == 1 and r0["iters"] == 40 and r0["updates"] >= 1
    with pytest.raises(ValueError):
        oracle.cg_mixed(dims, u, 0.1, 1e-10, 10, b, delta=1.5)


@pytest.mark.parametrize("n", [1, 17, 4096, 4097, 3 * 4096 + 17])
def test_fp32_inner_product_over_several_blocks_and_a_ragged_tail(n):
    """oracle.dot_re_f supplies every alpha, beta and update decision of oracle.cg_mixed (the
    sums) and adds in fixed 4096-element blocks like dot_re; the 16^4 and larger mixed runs (and the stored
    cfgN_mixed counts) go through the block loop.  Pinned against numpy's own product of the SAME fp32-rounded
    numbers -- exactly representable in fp64, so only the order of the additions differs -- at one element,
    under one block, one block exactly, one block + 1, and several blocks + a ragged tail."""
    rng = np.random.default_rng(2200 + n)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    a32 = a.astype(np.complex64).astype(np.complex128)
    b32 = b.astype(np.complex64).astype(np.complex128)
    scale = np.linalg.norm(a32) * np.linalg.norm(b32)
    want = np.vdot(a32, b32).real
    assert abs(oracle.dot_re_f(a, b) - want) <= 1e-14 * scale
    assert abs(oracle.dot_re_f(a, a) - np.linalg.norm(a32) ** 2) <= 1e-14 * scale
    # it really rounds to fp32 first: the fp64 product of the unrounded numbers is ~1e-8 away, not 1e-16
    if n >= 17:
        assert abs(oracle.dot_re_f(a, a) - np.linalg.norm(a) ** 2) > 1e-10 * np.linalg.norm(a) ** 2
    # every block counts, the last one included: a vector that is zero except in its last element
    e = np.zeros(n, complex)
    e[-1] = 3.0 - 4.0j
    assert oracle.dot_re_f(e, e) == 25.0
    assert oracle.dot_re_f(e, 1j * e) == 0.0


def test_mixed_cg_on_a_system_longer_than_one_block():
    """BASELINE.json config 2 (16^4: 98 304 complex per vector = 24 blocks of the inner products): the mixed
    oracle against the plain fp64 oracle CG (pinned by P7 and the residual tests) within the DESIGN.md 9.3
    bound, and its reported residual against one retaken here in numpy from the fp64 operator."""
    c, u, b = synth.config_inputs(2)
    dims, mass, tol = c["dims"], c["param"], c["tol"]
    want = oracle.cg(dims, STAGGERED, u, mass, tol, 20000, b)
    r = oracle.cg_mixed(dims, u, mass, tol, 20000, b)
    assert r["status"] == 0 and r["updates"] >= 2
    res = np.linalg.norm(b - oracle.apply_MdagM(dims, STAGGERED, u, mass, r["x"])) / np.linalg.norm(b)
    assert res <= tol and abs(res - r["true_residual"]) <= 1e-6 * res
    bound = 2 * tol * np.linalg.norm(b) / mass ** 2 / np.linalg.norm(want["x"])
    assert rel(r["x"], want["x"]) <= min(bound, 1e-8)
    assert want["iters"] <= r["iters"] + 2 and r["iters"] <= 1.25 * want["iters"] + 10
