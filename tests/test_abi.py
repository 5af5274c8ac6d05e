"""Host-side checks of the C-ABI library (no GPU): it loads, exports every symbol
include/lqcd.h declares, validates arguments, and never computes without a device."""
import ctypes

import pytest
import torch

import paper_1311_2719_b200 as pkg
from paper_1311_2719_b200 import lqcd


def test_library_exports_every_declared_symbol():
    names = lqcd.exported_symbols()
    assert {"lqcd_create", "lqcd_destroy", "lqcd_workspace_bytes", "lqcd_set_workspace", "lqcd_load_gauge",
            "lqcd_get_tables", "lqcd_dslash", "lqcd_apply_MdagM", "lqcd_cg_solve", "lqcd_last_error",
            "lqcd_congrad_host"} <= set(names)
    lib = ctypes.CDLL(lqcd.library_path())
    for n in names:
        assert hasattr(lib, n), n


def test_package_lazy_attributes():
    assert pkg.STAGGERED == 0 and pkg.WILSON == 1 and pkg.EVEN == 0 and pkg.ODD == 1
    assert pkg.Lattice is lqcd.Lattice


@pytest.mark.parametrize("dims,code", [((3, 4, 4, 4), -1), ((4, 4, 4, 0), -1), ((4, 4, 5, 4), -1),
                                       ((2048, 2048, 2048, 2), -1)])
def test_create_rejects_bad_extents(dims, code):
    with pytest.raises(lqcd.LqcdError) as e:
        lqcd.Lattice(dims, lqcd.STAGGERED, device="cpu")
    assert e.value.code == code


def test_create_rejects_bad_fermion_type():
    with pytest.raises(lqcd.LqcdError) as e:
        lqcd.Lattice((4, 4, 4, 4), 7, device="cpu")
    assert e.value.code == -2


@pytest.mark.parametrize("dims,fermion", [((4, 4, 4, 4), 0), ((32, 32, 32, 32), 0), ((16, 16, 16, 32), 1),
                                          ((48, 48, 48, 96), 0), ((2, 2, 2, 2), 1)])
def test_workspace_size_covers_gauge_vectors_and_staging(dims, fermion):
    lat = lqcd.Lattice(dims, fermion, device="cpu")
    v = lat.volume
    nvec = 3 * v // 2 if fermion == 0 else 12 * v
    need = 2 * v * 576 + 5 * nvec * 16          # internal + staged gauge, r p t + staged b x
    if fermion == 0:
        need += v * 288 + 4 * nvec * 8           # fp32 links and xs rs ps ts of the mixed-precision solver
    got = lat.workspace_bytes()
    assert need <= got <= need + 4 * 1024 * 1024 + v
    lat.close()


def test_compute_calls_need_workspace_and_never_fall_back():
    lat = lqcd.Lattice((4, 4, 4, 4), lqcd.STAGGERED, device="cpu")
    lib = lqcd.load_library()
    buf = (ctypes.c_double * 16)()
    assert lib.lqcd_dslash(lat._ctx, 0, buf, buf) == -3            # LQCD_ESTATE: no workspace
    assert lib.lqcd_load_gauge(lat._ctx, buf) == -3
    it, res = ctypes.c_int(), ctypes.c_double()
    assert lib.lqcd_cg_solve(lat._ctx, 0.1, 1e-10, 10, buf, buf, ctypes.byref(it), ctypes.byref(res)) == -3
    assert b"workspace" in lib.lqcd_last_error(lat._ctx)
    if not torch.cuda.is_available():
        # a host pointer as "workspace": the library must refuse for lack of a device, not compute
        big = ctypes.create_string_buffer(lat.workspace_bytes() + 512)
        addr = (ctypes.addressof(big) + 255) // 256 * 256
        assert lib.lqcd_set_workspace(lat._ctx, ctypes.c_void_p(addr), lat.workspace_bytes(), None) == -4
        with pytest.raises(lqcd.LqcdError):
            lqcd.Lattice((4, 4, 4, 4), lqcd.STAGGERED, device="cuda:0")
    assert lib.lqcd_set_option(lat._ctx, 99, 0) == -2
    assert lib.lqcd_set_option(lat._ctx, lqcd.OPT_CG_MODE, lqcd.CG_SYNC) == 0
    lat.close()


def test_null_context_is_an_error_not_a_crash():
    lib = lqcd.load_library()
    assert lib.lqcd_destroy(None) == -2
    assert lib.lqcd_workspace_bytes(None) == 0
    assert lib.lqcd_dslash(None, 0, None, None) == -2
