"""Host side of the time-slab decomposition (include/lqcd_slab.h, paper_1311_2719_b200/slab.py), no GPU:
the ABI loads and validates, the slab bookkeeping is pinned against an independent statement of the
site ordering (tests/lattice_util.py), the oracle confirms that one time-slice per face is all a slab
needs, and the set-up exchange between ranks runs over gloo with world size 2."""
import ctypes
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

import oracle
from lattice_util import site_coordinates, site_index
from paper_1311_2719_b200 import lqcd, slab, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------ ABI
def test_slab_library_exports_every_declared_symbol():
    names = slab.exported_symbols()
    assert {"lqcd_slab_create", "lqcd_slab_set_memory", "lqcd_slab_connect", "lqcd_slab_load_gauge", "lqcd_slab_dslash",
            "lqcd_slab_apply_MdagM", "lqcd_slab_cg_solve", "lqcd_slab_cg_solve_group", "lqcd_slab_ipc_export",
            "lqcd_slab_ipc_open"} <= set(names)
    lib = ctypes.CDLL(lqcd.library_path())
    for n in names:
        assert hasattr(lib, n), n


def _create(dims, rank, nranks):
    lib = slab._lib()
    s = ctypes.c_void_p()
    rc = lib.lqcd_slab_create(ctypes.byref(s), *dims, rank, nranks)
    return lib, s, rc


@pytest.mark.parametrize("dims,rank,nranks,code", [
    ((4, 4, 4, 12), 0, 4, -1),    # T = 3 is odd
    ((4, 4, 4, 4), 0, 4, -1),     # T = 1
    ((4, 4, 4, 6), 0, 4, -1),     # 6 % 4
    ((4, 3, 4, 8), 0, 2, -1),     # odd extent
    ((4, 4, 4, 8), 2, 2, -2),     # rank out of range
    ((4, 4, 4, 8), 0, 0, -2),
    ((4, 4, 4, 64), 0, 32, -2),   # more than LQCD_SLAB_MAX_RANKS
])
def test_slab_create_rejects(dims, rank, nranks, code):
    _, s, rc = _create(dims, rank, nranks)
    assert rc == code and not s.value


@pytest.mark.parametrize("dims,nranks", [((4, 4, 4, 8), 2), ((32, 32, 32, 32), 8), ((48, 48, 48, 96), 8)])
def test_slab_memory_sizes(dims, nranks):
    lib, s, rc = _create(dims, 1, nranks)
    assert rc == 0
    v_local = dims[0] * dims[1] * dims[2] * (dims[3] // nranks)
    sh = slab.half_slice(dims)
    need = v_local * 576 + 18 * sh * 16 + 3 * (3 * v_local // 2) * 16     # links, ghost links, r p t
    need += v_local * 288 + 18 * sh * 8 + 4 * (3 * v_local // 2) * 8      # fp32 copies of the mixed solver: links, ghost links, x r p t
    got = lib.lqcd_slab_workspace_bytes(s)
    assert need <= got <= need + 2 * 1024 * 1024 + v_local
    faces = 2 * 2 * 3 * sh * 16                                           # two buffers x two faces
    assert faces <= lib.lqcd_slab_mailbox_bytes(s) <= faces + 4096
    # no memory, no peers: compute calls are state errors, never a computation
    buf = (ctypes.c_double * 16)()
    assert lib.lqcd_slab_dslash(s, 0, buf, buf) == -3
    assert lib.lqcd_slab_load_gauge(s, buf, buf) == -3
    it, res = ctypes.c_int(), ctypes.c_double()
    assert lib.lqcd_slab_cg_solve(s, 0.1, 1e-10, 5, buf, buf, ctypes.byref(it), ctypes.byref(res)) == -3
    assert b"memory not set" in lib.lqcd_slab_last_error(s)
    arr = (ctypes.c_void_p * 1)(s.value)
    ptrs = (ctypes.c_void_p * 1)(ctypes.addressof(buf))
    assert lib.lqcd_slab_dslash_group(arr, 1, 0, ptrs, ptrs) == -2        # a group of 1 for a slab of rank 1 of n
    assert lib.lqcd_slab_set_option(s, 99, 0) == -2
    assert lib.lqcd_slab_set_option(s, slab.OPT_RECONSTRUCT, 12) == 0
    if not torch.cuda.is_available():
        big = ctypes.create_string_buffer(4096)
        addr = (ctypes.addressof(big) + 255) // 256 * 256
        assert lib.lqcd_slab_set_memory(s, ctypes.c_void_p(addr), 1 << 40, ctypes.c_void_p(addr), 1 << 40, None) == -4
        with pytest.raises(lqcd.LqcdError):
            slab.Slab(dims, 0, nranks)
    assert lib.lqcd_slab_destroy(s) == 0
    assert lib.lqcd_slab_destroy(None) == -2 and lib.lqcd_slab_workspace_bytes(None) == 0


# ------------------------------------------------------------------ bookkeeping against the site ordering
def _slab_sites_global_index(dims, rank, nranks):
    """g-index in the GLOBAL lattice of every site of the LOCAL lattice, in local canonical order."""
    ld = slab.local_dims(dims, nranks)
    x = site_coordinates(ld).copy()
    x[:, 3] += rank * ld[3]
    return site_index(dims, x)


@pytest.mark.parametrize("dims,nranks", [((4, 4, 4, 4), 2), ((4, 2, 6, 8), 4), ((6, 4, 2, 12), 3), ((2, 2, 2, 4), 1)])
def test_slab_rows_are_the_sites_of_the_time_slab(dims, nranks):
    v = synth.volume(dims)
    vh = v // 2
    u = torch.arange(v * 36, dtype=torch.float64).reshape(v, 4, 3, 3).to(torch.complex128)
    vec = torch.arange(3 * vh, dtype=torch.float64).reshape(3, vh).to(torch.complex128)
    parts = []
    for rank in range(nranks):
        g = _slab_sites_global_index(dims, rank, nranks)
        vl = g.shape[0] // 2
        assert torch.equal(slab.local_gauge(u, dims, rank, nranks), u[torch.from_numpy(g)])
        assert (g[:vl] < vh).all() and (g[vl:] >= vh).all()              # local parity = global parity
        part = slab.local_vector(vec, dims, rank, nranks)
        assert torch.equal(part, vec[:, torch.from_numpy(g[:vl])])
        parts.append(part)
        # u3_below: U_3 on the slice under the slab, both parities, in the order of a local time-slice
        sh = slab.half_slice(dims)
        ld1 = (dims[0], dims[1], dims[2], 2)                               # a 2-slice lattice gives the in-slice order
        x = site_coordinates(ld1).copy()
        tb = (rank * (dims[3] // nranks) - 1) % dims[3]
        below = []
        for parity in (0, 1):
            # sites of global parity `parity` on slice tb, ordered by their in-slice half index
            sel = x[(x[:, 3] == 0)]
            sel = sel.copy()
            sel[:, 3] = tb
            gi = site_index(dims, sel)
            gi = np.sort(gi[(gi >= vh) == bool(parity)])
            assert gi.shape[0] == sh
            below.append(u[torch.from_numpy(gi), 3])
        assert torch.equal(slab.u3_below_from_global(u, dims, rank, nranks), torch.stack(below))
        # the top U_3 slice of the rank below is the same thing
        lo = (rank - 1) % nranks
        assert torch.equal(slab.u3_top_slice(slab.local_gauge(u, dims, lo, nranks), dims, nranks),
                           slab.u3_below_from_global(u, dims, rank, nranks))
    assert torch.equal(slab.gather_vector(parts), vec)
    assert slab.neighbours(0, nranks) == ((nranks - 1) % nranks, 1 % nranks)


def test_slab_extent_rules():
    assert slab.slab_extent((4, 4, 4, 8), 2) == 4 and slab.slab_extent((4, 4, 4, 8), 4) == 2
    for dims, n in (((4, 4, 4, 8), 8), ((4, 4, 4, 12), 4), ((4, 4, 4, 8), 3), ((4, 4, 4, 8), 0), ((4, 4, 4, 64), 32)):
        with pytest.raises(ValueError):
            slab.slab_extent(dims, n)


def test_oracle_one_time_slice_per_face_is_all_a_slab_needs():
    """D is nearest-neighbour: the hopping term on a slab's sites is unchanged when the input vector is
    zeroed everywhere except on the slab and on the one time-slice on either side of it."""
    dims, nranks = (4, 4, 4, 8), 4
    vh, sh, T = synth.volume(dims) // 2, slab.half_slice(dims), 2
    u = synth.gauge_field(dims, "haar", 91)
    vin = synth.vector((3, vh), 92)
    full = oracle.dslash(dims, 0, u, 1, vin)
    for rank in range(nranks):
        keep = np.zeros(vh, bool)
        for t in range(rank * T - 1, (rank + 1) * T + 1):
            tt = t % dims[3]
            keep[tt * sh:(tt + 1) * sh] = True
        cut = np.where(keep[None, :], vin, 0.0)
        e0, e1 = slab.site_range(dims, rank, nranks)
        assert np.array_equal(oracle.dslash(dims, 0, u, 1, cut)[:, e0:e1], full[:, e0:e1])
        # ... and one slice less on either side is not enough
        keep[((rank * T - 1) % dims[3]) * sh:((rank * T - 1) % dims[3] + 1) * sh] = False
        cut = np.where(keep[None, :], vin, 0.0)
        assert not np.array_equal(oracle.dslash(dims, 0, u, 1, cut)[:, e0:e1], full[:, e0:e1])


# ------------------------------------------------------------------ two ranks over gloo
def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_1311_2719_b200 import slab as sl, synth as sy
    from paper_1311_2719_b200.ranks import Ranks
    r = Ranks(backend="gloo")
    dims = (4, 4, 4, 8)
    u = torch.from_numpy(sy.gauge_field(dims, "random_su3", 17))          # every rank can build the global field
    u_local = sl.local_gauge(u, dims, r.rank, r.world)
    got = sl.exchange_u3_below(u_local, dims, r.rank, r.world)            # what arrives from the rank below
    ok_u3 = torch.equal(got, sl.u3_below_from_global(u, dims, r.rank, r.world))
    # the faces a Dslash needs, moved the same way: my top slice is the upper rank's ghost_lo
    v = torch.from_numpy(sy.vector((3, sy.volume(dims) // 2), 18))
    mine = sl.local_vector(v, dims, r.rank, r.world)
    sh = sl.half_slice(dims)
    below, above = sl.neighbours(r.rank, r.world)
    ghost_lo = torch.empty(3, sh, dtype=torch.complex128)
    ops = [dist.P2POp(dist.isend, mine[:, -sh:].contiguous(), above), dist.P2POp(dist.irecv, ghost_lo, below)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    tb = (r.rank * (dims[3] // r.world) - 1) % dims[3]
    ok_face = torch.equal(ghost_lo, v[:, tb * sh:(tb + 1) * sh])
    gathered = [torch.empty_like(mine) for _ in range(r.world)]
    dist.all_gather(gathered, mine)
    ok_gather = torch.equal(sl.gather_vector(gathered), v)
    r.barrier()
    r.close()
    out.put(dict(rank=rank, ok_u3=ok_u3, ok_face=ok_face, ok_gather=ok_gather, below=below, above=above))


def test_two_ranks_gloo_slab_setup_exchange():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(i, 2, port, q)) for i in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=180) for _ in procs), key=lambda d: d["rank"])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for g in got:
        assert g["ok_u3"] and g["ok_face"] and g["ok_gather"]
        assert g["below"] == g["above"] == 1 - g["rank"]
