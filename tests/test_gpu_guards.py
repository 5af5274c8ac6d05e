"""Out-of-bounds WRITES of the CUDA path, caught with guard bands (compute-sanitizer is not available on
the GPU pool): every output vector sits between two bands of a known bit pattern inside one allocation;
after the call the bands must be untouched and the payload must match the oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_1311_2719_b200 import synth

pytestmark = pytest.mark.gpu

GUARD = 4096          # complex numbers on either side
PATTERN = complex(-1234.5, 6789.25)


def guarded(shape):
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * GUARD,), PATTERN, dtype=torch.complex128, device="cuda")
    return buf, buf[GUARD:GUARD + n].view(*shape)


def intact(buf):
    return bool((buf[:GUARD] == PATTERN).all().item()) and bool((buf[-GUARD:] == PATTERN).all().item())


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 8), (10, 6, 6, 4), (8, 8, 8, 8)])
def test_staggered_outputs_stay_inside_their_vectors(dims, recon):
    from paper_1311_2719_b200 import lqcd
    u = synth.gauge_field(dims, "haar", 301)
    b = synth.source(dims, "staggered", 302)
    with lqcd.Lattice(dims, lqcd.STAGGERED) as lat:
        lat.set_option(lqcd.OPT_RECONSTRUCT, recon)
        lat.load_gauge(torch.from_numpy(u).cuda())
        bd = torch.from_numpy(b).cuda()
        for parity in (0, 1):
            buf, out = guarded(lat.vector_shape)
            lat.dslash(parity, bd, out)
            torch.cuda.synchronize()
            assert intact(buf) and rel(out.cpu().numpy(), oracle.dslash(dims, 0, u, parity, b)) <= 1e-13
        buf, out = guarded(lat.vector_shape)
        lat.apply_MdagM(0.1, bd, out)
        torch.cuda.synchronize()
        assert intact(buf) and rel(out.cpu().numpy(), oracle.apply_MdagM(dims, 0, u, 0.1, b)) <= 1e-13
        want = oracle.cg(dims, 0, u, 0.1, 1e-10, 5000, b)
        buf, x = guarded(lat.vector_shape)
        lat.cg_solve(0.1, 1e-10, 5000, bd, x)
        assert intact(buf) and rel(x.cpu().numpy(), want["x"]) <= 1e-9
        buf, x = guarded(lat.vector_shape)
        lat.cg_solve_mixed(0.1, 1e-10, 5000, bd, x)
        assert intact(buf) and rel(x.cpu().numpy(), want["x"]) <= 1e-8


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 2, 6, 4), (4, 4, 4, 8)])
def test_wilson_outputs_stay_inside_their_vectors(dims):
    from paper_1311_2719_b200 import lqcd
    u = synth.gauge_field(dims, "smooth", 303)
    b = synth.source(dims, "wilson", 304)
    with lqcd.Lattice(dims, lqcd.WILSON) as lat:
        lat.load_gauge(torch.from_numpy(u).cuda())
        bd = torch.from_numpy(b).cuda()
        buf, out = guarded(lat.vector_shape)
        out.zero_()
        lat.dslash(1, bd, out)
        torch.cuda.synchronize()
        assert intact(buf) and rel(out.cpu().numpy(), oracle.dslash(dims, 1, u, 1, b)) <= 1e-13
        want = oracle.cg(dims, 1, u, 0.12, 1e-10, 5000, b)
        buf, x = guarded(lat.vector_shape)
        lat.cg_solve(0.12, 1e-10, 5000, bd, x)
        assert intact(buf) and rel(x.cpu().numpy(), want["x"]) <= 1e-9
        weo = oracle.wilson_solve_eo(dims, u, 0.12, 1e-10, 5000, b)
        buf, x = guarded(lat.vector_shape)
        lat.wilson_solve_eo(0.12, 1e-10, 5000, bd, x)
        assert intact(buf) and rel(x.cpu().numpy(), weo["x"]) <= 1e-9


@pytest.mark.parametrize("dims,nranks", [((4, 4, 4, 4), 2), ((4, 2, 6, 8), 4), ((8, 8, 8, 8), 2)])
def test_slab_outputs_stay_inside_their_vectors(dims, nranks):
    from paper_1311_2719_b200 import slab
    u = synth.gauge_field(dims, "haar", 305)
    b = synth.source(dims, "staggered", 306)
    g = slab.SlabGroup(dims, nranks)
    try:
        g.load_gauge_from_global(torch.from_numpy(u))
        bs = g.scatter(torch.from_numpy(b))
        pairs = [guarded(s.vector_shape) for s in g.slabs]
        g.dslash(1, bs, [p[1] for p in pairs])
        g.synchronize()
        got = slab.gather_vector([p[1].cpu() for p in pairs]).numpy()
        assert all(intact(p[0]) for p in pairs) and rel(got, oracle.dslash(dims, 0, u, 1, b)) <= 1e-13
        want = oracle.cg(dims, 0, u, 0.1, 1e-10, 5000, b)
        pairs = [guarded(s.vector_shape) for s in g.slabs]
        g.cg_solve(0.1, 1e-10, 5000, bs, [p[1] for p in pairs])
        got = slab.gather_vector([p[1].cpu() for p in pairs]).numpy()
        assert all(intact(p[0]) for p in pairs) and rel(got, want["x"]) <= 1e-9
    finally:
        g.close()
