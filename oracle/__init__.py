"""ctypes front end of the CPU oracle (oracle/lqcd_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the product package's binding and
the product never imports it.  Arrays are numpy complex128 / int32 in the canonical
layouts of SURVEY.md 8(b) (see the header of lqcd_oracle.c).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

STAGGERED, WILSON = 0, 1
EVEN, ODD = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lqcd_oracle.c")
_SO = os.path.join(_HERE, "liblqcd_oracle.so")
# No -ffast-math, no -march=native (the .so travels to another machine; no FMA
# contraction on baseline x86-64).  -fcx-limited-range = textbook complex product.
CFLAGS = ["-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared", "-Wall"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the shared object is missing or older than its source."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        P = ctypes.c_void_p
        L.oracle_tables.argtypes = [P, P, P, P]
        L.oracle_coords.argtypes = [P, P]
        L.oracle_dslash.argtypes = [P, ctypes.c_int, P, ctypes.c_int, P, P]
        L.oracle_dslash_sites.argtypes = [P, ctypes.c_int, P, ctypes.c_int, P, ctypes.c_long, P, P]
        L.oracle_wilson_M.argtypes = [P, P, ctypes.c_double, P, P]
        L.oracle_apply_MdagM.argtypes = [P, ctypes.c_int, P, ctypes.c_double, P, P]
        L.oracle_dot_re.argtypes = [P, P, ctypes.c_long]
        L.oracle_dot_re.restype = ctypes.c_double
        L.oracle_dot_re_f.argtypes = [P, P, ctypes.c_long]
        L.oracle_dot_re_f.restype = ctypes.c_double
        L.oracle_cg.argtypes = [P, ctypes.c_int, P, ctypes.c_double, ctypes.c_double, ctypes.c_int, P, P, P, P, P]
        L.oracle_stag_M.argtypes = [P, P, ctypes.c_double, P, P, P, P]
        L.oracle_stag_solve_full.argtypes = [P, P, ctypes.c_double, ctypes.c_double, ctypes.c_int, P, P, P, P, P, P]
        L.oracle_stag_dslash_f32.argtypes = [P, P, ctypes.c_int, P, P]
        L.oracle_cg_mixed.argtypes = [P, P, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int, P, P, P, P, P, P]
        L.oracle_wilson_Mhat.argtypes = [P, P, ctypes.c_double, ctypes.c_int, P, P]
        L.oracle_wilson_solve_eo.argtypes = [P, P, ctypes.c_double, ctypes.c_double, ctypes.c_int, P, P, P, P]
        L.oracle_num_threads.restype = ctypes.c_int
        L.oracle_set_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def _dims(dims):
    return np.asarray(dims, dtype=np.int32)


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _check(rc, what):
    if rc < 0:
        raise ValueError("%s failed with code %d" % (what, rc))
    return rc


def num_threads() -> int:
    return lib().oracle_num_threads()


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def volume(dims) -> int:
    return int(np.prod(np.asarray(dims, dtype=np.int64)))


def tables(dims):
    """(iup[4][V], idn[4][V], lex2eo[V]) int32."""
    v = volume(dims)
    d = _dims(dims)
    iup = np.empty((4, v), np.int32)
    idn = np.empty((4, v), np.int32)
    l2e = np.empty(v, np.int32)
    _check(lib().oracle_tables(_ptr(d), _ptr(iup), _ptr(idn), _ptr(l2e)), "oracle_tables")
    return iup, idn, l2e


def coords(dims):
    """x[g][mu] int32 for every canonical site index g."""
    v = volume(dims)
    d = _dims(dims)
    x = np.empty((v, 4), np.int32)
    _check(lib().oracle_coords(_ptr(d), _ptr(x)), "oracle_coords")
    return x


def _vec_shape(dims, fermion):
    v = volume(dims)
    return (3, v // 2) if fermion == STAGGERED else (4, 3, v)


def dslash(dims, fermion, u, out_parity, vin, out=None):
    """Bare hopping term.  Staggered: (3,Vh)->(3,Vh).  Wilson: full (4,3,V) in, writes the
    out_parity half of `out` (a zero-filled array is made if none is given)."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    vin = _c(vin, np.complex128)
    assert u.shape == (volume(dims), 4, 3, 3) and vin.shape == _vec_shape(dims, fermion)
    if out is None:
        out = np.zeros(_vec_shape(dims, fermion), np.complex128)
    _check(lib().oracle_dslash(_ptr(d), fermion, _ptr(u), out_parity, _ptr(vin), _ptr(out)), "oracle_dslash")
    return out


def dslash_sites(dims, fermion, u, out_parity, vin, e_list):
    """Hopping term at the listed half-lattice indices only: (n,3) or (n,4,3)."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    vin = _c(vin, np.complex128)
    e = _c(e_list, np.int64)
    out = np.empty((len(e), 3) if fermion == STAGGERED else (len(e), 4, 3), np.complex128)
    _check(lib().oracle_dslash_sites(_ptr(d), fermion, _ptr(u), out_parity, _ptr(vin), len(e), _ptr(e), _ptr(out)),
           "oracle_dslash_sites")
    return out


def wilson_M(dims, u, kappa, vin):
    d = _dims(dims)
    u = _c(u, np.complex128)
    vin = _c(vin, np.complex128)
    out = np.empty_like(vin)
    _check(lib().oracle_wilson_M(_ptr(d), _ptr(u), float(kappa), _ptr(vin), _ptr(out)), "oracle_wilson_M")
    return out


def apply_MdagM(dims, fermion, u, param, vin):
    d = _dims(dims)
    u = _c(u, np.complex128)
    vin = _c(vin, np.complex128)
    assert vin.shape == _vec_shape(dims, fermion)
    out = np.empty_like(vin)
    _check(lib().oracle_apply_MdagM(_ptr(d), fermion, _ptr(u), float(param), _ptr(vin), _ptr(out)), "oracle_apply_MdagM")
    return out


def dot_re(a, b) -> float:
    a = _c(a, np.complex128)
    b = _c(b, np.complex128)
    return lib().oracle_dot_re(_ptr(a), _ptr(b), a.size)


def dot_re_f(a, b) -> float:
    """Re<fl32(a), fl32(b)> accumulated in fp64: the inner product of the mixed-precision CG."""
    a = _c(a, np.complex128)
    b = _c(b, np.complex128)
    return lib().oracle_dot_re_f(_ptr(a), _ptr(b), a.size)


def cg(dims, fermion, u, param, tol, maxiter, b, history=False):
    """Returns dict(x, iters, true_residual, status[, rr_history])."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    b = _c(b, np.complex128)
    assert b.shape == _vec_shape(dims, fermion)
    x = np.empty_like(b)
    it = ctypes.c_int(0)
    res = ctypes.c_double(0.0)
    hist = np.zeros(maxiter + 1, np.float64) if history else None
    rc = _check(lib().oracle_cg(_ptr(d), fermion, _ptr(u), float(param), float(tol), int(maxiter), _ptr(b), _ptr(x),
                                ctypes.byref(it), ctypes.byref(res), _ptr(hist) if history else None), "oracle_cg")
    out = dict(x=x, iters=it.value, true_residual=res.value, status=rc)
    if history:
        out["rr_history"] = hist[: it.value + 1]
    return out


def stag_M(dims, u, mass, in_e, in_o):
    """(M in)_e, (M in)_o with M = m + D on a full-lattice staggered vector given as its two halves."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    in_e = _c(in_e, np.complex128)
    in_o = _c(in_o, np.complex128)
    assert in_e.shape == _vec_shape(dims, STAGGERED) and in_o.shape == in_e.shape
    out_e, out_o = np.empty_like(in_e), np.empty_like(in_o)
    _check(lib().oracle_stag_M(_ptr(d), _ptr(u), float(mass), _ptr(in_e), _ptr(in_o), _ptr(out_e), _ptr(out_o)),
           "oracle_stag_M")
    return out_e, out_o


def stag_solve_full(dims, u, mass, tol, maxiter, b_e, b_o):
    """M x = b on the full lattice by even-odd reduction: dict(x_e, x_o, iters, true_residual, status)."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    b_e = _c(b_e, np.complex128)
    b_o = _c(b_o, np.complex128)
    assert b_e.shape == _vec_shape(dims, STAGGERED) and b_o.shape == b_e.shape
    x_e, x_o = np.empty_like(b_e), np.empty_like(b_o)
    it = ctypes.c_int(0)
    res = ctypes.c_double(0.0)
    rc = _check(lib().oracle_stag_solve_full(_ptr(d), _ptr(u), float(mass), float(tol), int(maxiter), _ptr(b_e),
                                             _ptr(b_o), _ptr(x_e), _ptr(x_o), ctypes.byref(it), ctypes.byref(res)),
                "oracle_stag_solve_full")
    return dict(x_e=x_e, x_o=x_o, iters=it.value, true_residual=res.value, status=rc)


def stag_dslash_f32(dims, u, out_parity, vin):
    """The staggered hopping term evaluated in fp32 on fl32(u), fl32(vin); returned widened to complex128."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    vin = _c(vin, np.complex128)
    assert vin.shape == _vec_shape(dims, STAGGERED)
    out = np.empty_like(vin)
    _check(lib().oracle_stag_dslash_f32(_ptr(d), _ptr(u), int(out_parity), _ptr(vin), _ptr(out)), "oracle_stag_dslash_f32")
    return out


def cg_mixed(dims, u, mass, tol, maxiter, b, delta=0.1, history=False):
    """Mixed-precision CG with reliable updates: dict(x, iters, updates, true_residual, status[, rr_history])."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    b = _c(b, np.complex128)
    assert b.shape == _vec_shape(dims, STAGGERED)
    x = np.empty_like(b)
    it, nu = ctypes.c_int(0), ctypes.c_int(0)
    res = ctypes.c_double(0.0)
    hist = np.zeros(maxiter + 1, np.float64) if history else None
    rc = _check(lib().oracle_cg_mixed(_ptr(d), _ptr(u), float(mass), float(tol), float(delta), int(maxiter), _ptr(b),
                                      _ptr(x), ctypes.byref(it), ctypes.byref(nu), ctypes.byref(res),
                                      _ptr(hist) if history else None), "oracle_cg_mixed")
    out = dict(x=x, iters=it.value, updates=nu.value, true_residual=res.value, status=rc)
    if history:
        out["rr_history"] = hist[: it.value + 1]
    return out


def wilson_Mhat(dims, u, kappa, vin, dagger=False):
    """Schur complement Mhat = 1 - kappa^2 D_eo D_oe (or its adjoint) on the even half of a full-lattice
    Wilson vector; the odd half of the result is zero."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    vin = _c(vin, np.complex128)
    assert vin.shape == _vec_shape(dims, WILSON)
    out = np.empty_like(vin)
    _check(lib().oracle_wilson_Mhat(_ptr(d), _ptr(u), float(kappa), int(bool(dagger)), _ptr(vin), _ptr(out)),
           "oracle_wilson_Mhat")
    return out


def wilson_solve_eo(dims, u, kappa, tol, maxiter, b):
    """M x = b (M = 1 - kappa D_W) by even-odd preconditioning: dict(x, iters, true_residual, status)."""
    d = _dims(dims)
    u = _c(u, np.complex128)
    b = _c(b, np.complex128)
    assert b.shape == _vec_shape(dims, WILSON)
    x = np.empty_like(b)
    it = ctypes.c_int(0)
    res = ctypes.c_double(0.0)
    rc = _check(lib().oracle_wilson_solve_eo(_ptr(d), _ptr(u), float(kappa), float(tol), int(maxiter), _ptr(b), _ptr(x),
                                             ctypes.byref(it), ctypes.byref(res)), "oracle_wilson_solve_eo")
    return dict(x=x, iters=it.value, true_residual=res.value, status=rc)
