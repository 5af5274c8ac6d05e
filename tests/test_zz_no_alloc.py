"""lqcd_cg_init_noalloc (include/lqcd_noalloc.h): the S6 pass of the conjugate gradient for callers that cannot
allocate device memory when they need it -- a simulation whose fields already fill the GPU, a plug-in under a
framework that owns the allocator, a trajectory that cannot take cudaMalloc's device-wide stall.  Its reduction
scratch is a fixed array inside the library, shared by every call on a GPU, so the thing to check is that a call
gives the right answer whatever the PREVIOUS call left in that array: two calls in a row, different vectors and
lengths, each against the library's ordinary path (lqcd_cg_solve's S6 kernel, scratch in the caller's workspace).

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  The GPU test builds everything it needs itself, so it passes alone in a fresh process (where
its first call is also the one that looks up the array's device address) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_1311_2719_b200 import lqcd, noalloc, synth

TOL = 1e-13   # the relative tolerance of the fp64 parity tests (tests/test_gpu_parity.py DSLASH_TOL)


def test_header_symbols_are_exported_and_the_limit_is_the_documented_one():
    lib = ctypes.CDLL(lqcd.library_path())
    for name in ("lqcd_cg_init_noalloc", "lqcd_noalloc_max_complex", "lqcd_noalloc_last_error"):
        assert hasattr(lib, name), name
    assert noalloc.max_complex() == 4096 * 8192 == 33_554_432


def test_refusals_happen_before_anything_touches_a_device():
    """Too long a vector, a null pointer, a misaligned pointer: refused on the host with a message, no launch
    (the pointers below are host memory; had a kernel been given them the GPU test after this would tell)."""
    lib = lqcd.load_library()
    buf = (ctypes.c_double * 8)()
    base = ctypes.addressof(buf)
    base += (-base) % 16
    p = ctypes.c_void_p(base)
    too_long = noalloc.max_complex() + 1
    assert lib.lqcd_cg_init_noalloc(p, p, p, p, too_long, p, None) == -5          # LQCD_ENOMEM
    msg = noalloc.last_error()
    assert str(too_long) in msg and "LQCD_NOALLOC_MAX_COMPLEX" in msg and "33554432" in msg
    assert lib.lqcd_cg_init_noalloc(p, None, p, p, 2, p, None) == -2                # LQCD_EARG: null vector
    assert lib.lqcd_cg_init_noalloc(p, p, p, p, 2, None, None) == -2                # null bb
    assert lib.lqcd_cg_init_noalloc(ctypes.c_void_p(base + 8), p, p, p, 2, p, None) == -2   # complex fp64 needs 16
    assert "aligned" in noalloc.last_error()


# (lattice, seed): 25 920 complex = 6 full tiles of 4096 + a ragged one; then 4 608 = 1 tile + 512, so the second
# call finds five stale partial sums of the first beyond the two it writes; then the first length again.
CALLS = [((12, 12, 12, 10), 31), ((8, 8, 8, 6), 32), ((12, 12, 12, 10), 33)]
GUARD = 64


def _existing_path(dims, b):
    """<b,b> and x of the ordinary path: lqcd_cg_solve with maxiter = 0 runs exactly its S6 kernel (x = 0,
    history[0] = <b,b>) with the reduction scratch in the workspace torch allocated."""
    u = synth.gauge_field(dims, "haar", 5)
    with lqcd.Lattice(dims, lqcd.STAGGERED) as lat:
        lat.load_gauge(torch.from_numpy(u).cuda())
        x, it, _, status = lat.cg_solve(0.1, 1e-10, 0, b)
        assert it == 0 and status == lqcd.MAXITER
        return float(lat.cg_history()[0]), x.cpu()


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    bb = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    seen = []
    for dims, seed in CALLS:
        b = torch.from_numpy(synth.source(dims, "staggered", seed)).cuda()
        n = b.numel()
        # the caller's output buffers, pre-filled so that an element the kernel skipped, or one it wrote
        # past the end, shows
        outs = [torch.full((n + GUARD,), complex(float("nan"), 7.0), dtype=torch.complex128, device="cuda")
                for _ in range(3)]
        x, r, p = (o[:n].view(b.shape) for o in outs)
        noalloc.cg_init_noalloc(b, x, r, p, bb)
        got = float(bb.cpu()[0])

        want_bb, want_x = _existing_path(dims, b)
        assert abs(got - want_bb) <= TOL * want_bb, (dims, got, want_bb)
        b_host = b.cpu().numpy()
        assert abs(got - np.vdot(b_host, b_host).real) <= TOL * want_bb
        assert torch.equal(x.cpu(), want_x) and not want_x.any()                       # x = 0, as the existing path
        assert torch.equal(r.cpu(), b.cpu()) and torch.equal(p.cpu(), b.cpu())         # copies are bit-exact
        for o in outs:                                                                 # nothing past the vector
            tail = o[n:].cpu()
            assert torch.isnan(tail.real).all() and (tail.imag == 7.0).all()
        seen.append(got)

    # the sum is deterministic: the same vector again, whatever ran in between, gives the same bits
    dims, seed = CALLS[0]
    b = torch.from_numpy(synth.source(dims, "staggered", seed)).cuda()
    x, r, p = (torch.empty_like(b) for _ in range(3))
    noalloc.cg_init_noalloc(b, x, r, p, bb)
    assert float(bb.cpu()[0]) == seen[0]

    # an empty vector is legal: nothing to write but <b,b> = 0
    e = torch.empty((3, 0), dtype=torch.complex128, device="cuda")
    noalloc.cg_init_noalloc(e, e.clone(), e.clone(), e.clone(), bb)
    assert float(bb.cpu()[0]) == 0.0
