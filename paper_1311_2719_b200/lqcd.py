"""Thin ctypes binding of include/lqcd.h -- argument marshalling only.

Every step of the path runs in the CUDA library; PyTorch is used for device memory, pinned host
memory and the stream.  If ``liblqcd_b200.so`` has not been built, importing this module raises
(there is no CPU fallback; ``python -m paper_1311_2719_b200.build`` or
``__graft_entry__.build()`` compiles it).

Tensors are ``torch.complex128`` in the canonical layouts of include/lqcd.h:
gauge (V,4,3,3); staggered vectors (3,Vh); Wilson vectors (4,3,V).
"""
from __future__ import annotations

import ctypes
import os
import re

import torch

STAGGERED, WILSON = 0, 1
EVEN, ODD = 0, 1
OK, MAXITER = 0, 1
CG_SYNC, CG_ASYNC, CG_GRAPH = 0, 1, 2
PATH_NONE, PATH_HOST_LOOP, PATH_PERSISTENT = 0, 1, 2
OPT_CG_MODE, OPT_CG_CHECK_EVERY, OPT_RECONSTRUCT, OPT_CONGRAD_PRECISION, OPT_F32_PAIRS, OPT_PERSISTENT, OPT_STAG_BLOCK = 0, 1, 2, 3, 4, 5, 6
OPT_PERSISTENT_CHUNK = 7

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
_SO = os.path.join(_HERE, "liblqcd_b200.so")
_HEADER = os.path.join(_ROOT, "include", "lqcd.h")


class LqcdError(RuntimeError):
    def __init__(self, code, message):
        super().__init__("lqcd error %d: %s" % (code, message))
        self.code = code


def library_path() -> str:
    return _SO


def exported_symbols() -> list[str]:
    """Every function include/lqcd.h declares (the header is the single list of entry points)."""
    text = open(_HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_[a-zA-Z0-9_]+)\s*\(", text)))


_lib = None


def load_library():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_SO):
        raise ImportError("CUDA library %s is missing: build it with `python -m paper_1311_2719_b200.build` "
                          "(there is no CPU fallback)" % _SO)
    L = ctypes.CDLL(_SO)
    P, I, D = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    L.lqcd_create.argtypes = [ctypes.POINTER(P), I, I, I, I, I]
    L.lqcd_destroy.argtypes = [P]
    L.lqcd_workspace_bytes.argtypes = [P]
    L.lqcd_workspace_bytes.restype = ctypes.c_size_t
    L.lqcd_set_workspace.argtypes = [P, P, ctypes.c_size_t, P]
    L.lqcd_set_option.argtypes = [P, I, I]
    L.lqcd_load_gauge.argtypes = [P, P]
    L.lqcd_get_tables.argtypes = [P, P, P, P]
    L.lqcd_dslash.argtypes = [P, I, P, P]
    L.lqcd_dslash_sweep.argtypes = [P, I, P, P, I]
    L.lqcd_apply_MdagM.argtypes = [P, D, P, P]
    L.lqcd_cg_solve.argtypes = [P, D, D, I, P, P, ctypes.POINTER(I), ctypes.POINTER(D)]
    L.lqcd_cg_solve_mixed.argtypes = [P, D, D, I, D, P, P, ctypes.POINTER(I), ctypes.POINTER(I), ctypes.POINTER(D)]
    L.lqcd_stag_solve_full.argtypes = [P, D, D, I, P, P, P, P, ctypes.POINTER(I), ctypes.POINTER(D)]
    L.lqcd_wilson_eo_MdagM.argtypes = [P, D, P, P]
    L.lqcd_wilson_solve_eo.argtypes = [P, D, D, I, P, P, ctypes.POINTER(I), ctypes.POINTER(D)]
    L.lqcd_congrad_host.argtypes = [P, P, D, D, I, P, P, ctypes.POINTER(I), ctypes.POINTER(D)]
    L.lqcd_dslash_host.argtypes = [P, I, P, P]
    L.lqcd_cg_history.argtypes = [P, P, I]
    L.lqcd_kernel_launches.argtypes = [P]
    L.lqcd_kernel_launches.restype = ctypes.c_longlong
    L.lqcd_last_cg_path.argtypes = [P]
    L.lqcd_last_error.argtypes = [P]
    L.lqcd_last_error.restype = ctypes.c_char_p
    _lib = L
    return L


load_library()  # fail loudly at import time if the extension is missing


def _cptr(t: torch.Tensor):
    return ctypes.c_void_p(t.data_ptr())


class Lattice:
    """One lqcd_ctx plus the PyTorch-owned workspace and stream it runs on."""

    def __init__(self, dims, fermion: int = STAGGERED, device="cuda:0", stream: torch.cuda.Stream | None = None):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        self.dims = tuple(int(d) for d in dims)
        self.fermion = int(fermion)
        rc = self._lib.lqcd_create(ctypes.byref(self._ctx), *self.dims, self.fermion)
        if rc != 0:
            self._ctx = ctypes.c_void_p()
            raise LqcdError(rc, "lqcd_create%r failed (extents must be even and >= 2)" % (self.dims,))
        self.volume = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self.half_volume = self.volume // 2
        self.vector_shape = (3, self.half_volume) if self.fermion == STAGGERED else (4, 3, self.volume)
        self.device = torch.device(device)
        self.workspace = None
        self.stream = None
        if self.device.type == "cuda":
            self._bind(stream)

    # ------------------------------------------------------------------ plumbing
    def _bind(self, stream):
        if not torch.cuda.is_available():
            raise LqcdError(-4, "no CUDA device (the CUDA path is the only path)")
        nbytes = self._lib.lqcd_workspace_bytes(self._ctx)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        self._check(self._lib.lqcd_set_workspace(self._ctx, ctypes.c_void_p(aligned), nbytes,
                                                 ctypes.c_void_p(self.stream.cuda_stream)))

    def _check(self, rc):
        if rc < 0:
            raise LqcdError(rc, self._lib.lqcd_last_error(self._ctx).decode())
        return rc

    def workspace_bytes(self) -> int:
        return self._lib.lqcd_workspace_bytes(self._ctx)

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            if self.stream is not None:
                self.stream.synchronize()
            self._lib.lqcd_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _vec(self, t: torch.Tensor, name="vector") -> torch.Tensor:
        if t.dtype != torch.complex128 or t.device != self.device or not t.is_contiguous():
            raise ValueError("%s must be a contiguous complex128 tensor on %s" % (name, self.device))
        if tuple(t.shape) != self.vector_shape:
            raise ValueError("%s has shape %r, expected %r" % (name, tuple(t.shape), self.vector_shape))
        return t

    def _sync_in(self):
        # work queued by torch on its current stream (allocations, H2D copies) must precede ours
        self.stream.wait_stream(torch.cuda.current_stream(self.device))

    def _sync_out(self):
        torch.cuda.current_stream(self.device).wait_stream(self.stream)

    def new_vector(self) -> torch.Tensor:
        return torch.empty(self.vector_shape, dtype=torch.complex128, device=self.device)

    def set_option(self, option: int, value: int):
        self._check(self._lib.lqcd_set_option(self._ctx, int(option), int(value)))

    def kernel_launches(self) -> int:
        return int(self._lib.lqcd_kernel_launches(self._ctx))

    def last_cg_path(self) -> int:
        """PATH_NONE / PATH_HOST_LOOP / PATH_PERSISTENT: the iteration loop the last CG call ran."""
        return int(self._lib.lqcd_last_cg_path(self._ctx))

    # ------------------------------------------------------------------ the calls of include/lqcd.h
    def load_gauge(self, u: torch.Tensor):
        if u.dtype != torch.complex128 or u.device != self.device or not u.is_contiguous() \
                or tuple(u.shape) != (self.volume, 4, 3, 3):
            raise ValueError("gauge field must be contiguous complex128 (V,4,3,3) on %s" % self.device)
        self._sync_in()
        self._check(self._lib.lqcd_load_gauge(self._ctx, _cptr(u)))
        u.record_stream(self.stream)
        self._sync_out()

    def tables(self):
        """(iup[4][V], idn[4][V], lex2eo[V]) as int32 CPU tensors, built on the device."""
        v = self.volume
        iup = torch.empty((4, v), dtype=torch.int32)
        idn = torch.empty((4, v), dtype=torch.int32)
        l2e = torch.empty((v,), dtype=torch.int32)
        self._check(self._lib.lqcd_get_tables(self._ctx, _cptr(iup), _cptr(idn), _cptr(l2e)))
        return iup, idn, l2e

    def dslash(self, out_parity: int, vin: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        self._vec(vin, "in")
        if out is None:
            out = torch.zeros_like(vin) if self.fermion == WILSON else torch.empty_like(vin)
        self._vec(out, "out")
        self._sync_in()
        self._check(self._lib.lqcd_dslash(self._ctx, int(out_parity), _cptr(vin), _cptr(out)))
        self._sync_out()
        return out

    def dslash_sweep(self, first_out_parity: int, a: torch.Tensor, b: torch.Tensor, reps: int) -> None:
        """`reps` back-to-back hopping terms enqueued natively, ping-pong a -> b -> a ... (timing only)."""
        self._vec(a, "a")
        self._vec(b, "b")
        self._sync_in()
        self._check(self._lib.lqcd_dslash_sweep(self._ctx, int(first_out_parity), _cptr(a), _cptr(b), int(reps)))

    def apply_MdagM(self, mass_or_kappa: float, vin: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        self._vec(vin, "in")
        if out is None:
            out = torch.empty_like(vin)
        self._vec(out, "out")
        self._sync_in()
        self._check(self._lib.lqcd_apply_MdagM(self._ctx, float(mass_or_kappa), _cptr(vin), _cptr(out)))
        self._sync_out()
        return out

    def cg_solve(self, mass_or_kappa: float, tol: float, maxiter: int, b: torch.Tensor, x: torch.Tensor | None = None):
        """Returns (x, iters, true_residual, status); status 0 = converged, 1 = maxiter reached."""
        self._vec(b, "b")
        if x is None:
            x = torch.empty_like(b)
        self._vec(x, "x")
        it = ctypes.c_int(0)
        res = ctypes.c_double(0.0)
        self._sync_in()
        rc = self._check(self._lib.lqcd_cg_solve(self._ctx, float(mass_or_kappa), float(tol), int(maxiter), _cptr(b),
                                                 _cptr(x), ctypes.byref(it), ctypes.byref(res)))
        self._sync_out()
        return x, it.value, res.value, rc

    def cg_solve_mixed(self, mass: float, tol: float, maxiter: int, b: torch.Tensor, x: torch.Tensor | None = None,
                       delta: float = 0.1):
        """fp32 inner CG with fp64 reliable updates: (x, iters, reliable_updates, true_residual, status)."""
        self._vec(b, "b")
        if x is None:
            x = torch.empty_like(b)
        self._vec(x, "x")
        it, nu = ctypes.c_int(0), ctypes.c_int(0)
        res = ctypes.c_double(0.0)
        self._sync_in()
        rc = self._check(self._lib.lqcd_cg_solve_mixed(self._ctx, float(mass), float(tol), int(maxiter), float(delta),
                                                       _cptr(b), _cptr(x), ctypes.byref(it), ctypes.byref(nu),
                                                       ctypes.byref(res)))
        self._sync_out()
        return x, it.value, nu.value, res.value, rc

    def stag_solve_full(self, mass: float, tol: float, maxiter: int, b_even: torch.Tensor, b_odd: torch.Tensor,
                        x_even: torch.Tensor | None = None, x_odd: torch.Tensor | None = None):
        """M x = b on the full lattice (M = m + D): returns (x_even, x_odd, iters, true_residual, status)."""
        self._vec(b_even, "b_even")
        self._vec(b_odd, "b_odd")
        x_even = torch.empty_like(b_even) if x_even is None else self._vec(x_even, "x_even")
        x_odd = torch.empty_like(b_odd) if x_odd is None else self._vec(x_odd, "x_odd")
        it = ctypes.c_int(0)
        res = ctypes.c_double(0.0)
        self._sync_in()
        rc = self._check(self._lib.lqcd_stag_solve_full(self._ctx, float(mass), float(tol), int(maxiter), _cptr(b_even),
                                                        _cptr(b_odd), _cptr(x_even), _cptr(x_odd), ctypes.byref(it),
                                                        ctypes.byref(res)))
        self._sync_out()
        return x_even, x_odd, it.value, res.value, rc

    def wilson_eo_MdagM(self, kappa: float, vin: torch.Tensor, out: torch.Tensor | None = None) -> torch.Tensor:
        """Even half of out = Mhat^+ Mhat (even half of vin); a fresh `out` has a zero odd half."""
        self._vec(vin, "in")
        if out is None:
            out = torch.zeros_like(vin)
        self._vec(out, "out")
        self._sync_in()
        self._check(self._lib.lqcd_wilson_eo_MdagM(self._ctx, float(kappa), _cptr(vin), _cptr(out)))
        self._sync_out()
        return out

    def wilson_solve_eo(self, kappa: float, tol: float, maxiter: int, b: torch.Tensor, x: torch.Tensor | None = None):
        """M x = b (M = 1 - kappa D_W) by even-odd preconditioning: (x, iters, true_residual, status)."""
        self._vec(b, "b")
        if x is None:
            x = torch.empty_like(b)
        self._vec(x, "x")
        it = ctypes.c_int(0)
        res = ctypes.c_double(0.0)
        self._sync_in()
        rc = self._check(self._lib.lqcd_wilson_solve_eo(self._ctx, float(kappa), float(tol), int(maxiter), _cptr(b),
                                                        _cptr(x), ctypes.byref(it), ctypes.byref(res)))
        self._sync_out()
        return x, it.value, res.value, rc

    def congrad_host(self, u_host: torch.Tensor, mass_or_kappa: float, tol: float, maxiter: int, b_host: torch.Tensor,
                     x_host: torch.Tensor | None = None):
        """The paper's congrad with its data region: HOST tensors in, HOST tensor out."""
        for t, shape, name in ((u_host, (self.volume, 4, 3, 3), "u_host"), (b_host, self.vector_shape, "b_host")):
            if t.device.type != "cpu" or t.dtype != torch.complex128 or not t.is_contiguous() or tuple(t.shape) != shape:
                raise ValueError("%s must be a contiguous complex128 CPU tensor of shape %r" % (name, shape))
        if x_host is None:
            x_host = torch.empty(self.vector_shape, dtype=torch.complex128).pin_memory()
        it = ctypes.c_int(0)
        res = ctypes.c_double(0.0)
        rc = self._check(self._lib.lqcd_congrad_host(self._ctx, _cptr(u_host), float(mass_or_kappa), float(tol),
                                                     int(maxiter), _cptr(b_host), _cptr(x_host), ctypes.byref(it),
                                                     ctypes.byref(res)))
        return x_host, it.value, res.value, rc

    def dslash_host(self, out_parity: int, in_host: torch.Tensor, out_host: torch.Tensor | None = None):
        if out_host is None:
            out_host = torch.empty(self.vector_shape, dtype=torch.complex128).pin_memory()
        self._check(self._lib.lqcd_dslash_host(self._ctx, int(out_parity), _cptr(in_host), _cptr(out_host)))
        return out_host

    def cg_history(self, capacity: int = 65536) -> torch.Tensor:
        h = torch.empty((capacity,), dtype=torch.float64)
        n = self._check(self._lib.lqcd_cg_history(self._ctx, _cptr(h), capacity))
        return h[:n].clone()
