"""ctypes binding of include/lqcd_noalloc.h -- argument marshalling only.

``cg_init_noalloc`` is for callers that cannot allocate device memory when they need the kernel: a
simulation whose fields already fill the GPU, a plug-in under a framework that owns the allocator, a
trajectory with other streams in flight that a ``cudaMalloc`` would stall.  So this wrapper allocates
nothing either: the caller passes EVERY buffer, outputs and the one-element ``bb`` included.  The
reduction scratch is a fixed 64 KiB array inside the library (one per GPU, shared by all calls, vectors of
at most ``max_complex()`` = 33 554 432 complex numbers); calls that overlap on the GPU race on it, and the
first call on each device (which looks the array's address up) belongs at set-up time, before any stream
capture.  Details: the header.
"""
from __future__ import annotations

import ctypes

import torch

from . import lqcd

_lib = lqcd.load_library()   # raises if the CUDA library has not been built: there is no fallback
_lib.lqcd_cg_init_noalloc.argtypes = [ctypes.c_void_p] * 4 + [ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p]
_lib.lqcd_cg_init_noalloc.restype = ctypes.c_int
_lib.lqcd_noalloc_max_complex.argtypes = []
_lib.lqcd_noalloc_max_complex.restype = ctypes.c_size_t
_lib.lqcd_noalloc_last_error.argtypes = []
_lib.lqcd_noalloc_last_error.restype = ctypes.c_char_p


def max_complex() -> int:
    """Longest vector (in complex numbers) the static scratch can serve."""
    return int(_lib.lqcd_noalloc_max_complex())


def last_error() -> str:
    return _lib.lqcd_noalloc_last_error().decode()


def cg_init_noalloc(b: torch.Tensor, x: torch.Tensor, r: torch.Tensor, p: torch.Tensor, bb: torch.Tensor,
                    stream: torch.cuda.Stream | None = None) -> None:
    """p = r = b, x = 0, bb[0] = <b,b>, enqueued on `stream` (default: torch's current stream
    of b's device).  All tensors are the caller's: b, x, r, p contiguous complex128 of one shape on one CUDA
    device, bb a float64 tensor with one element on the same device.  Nothing is allocated, nothing is
    synchronised; raises lqcd.LqcdError on a refused call (vector too long: code -5)."""
    for t, name in ((b, "b"), (x, "x"), (r, "r"), (p, "p")):
        if t.dtype != torch.complex128 or not t.is_cuda or not t.is_contiguous() or t.shape != b.shape \
                or t.device != b.device:
            raise ValueError("%s must be a contiguous complex128 CUDA tensor shaped and placed like b" % name)
    if bb.dtype != torch.float64 or bb.numel() != 1 or bb.device != b.device:
        raise ValueError("bb must be a one-element float64 tensor on %s" % b.device)
    with torch.cuda.device(b.device):   # the library looks its scratch up on the CURRENT device
        s = stream if stream is not None else torch.cuda.current_stream(b.device)
        rc = _lib.lqcd_cg_init_noalloc(b.data_ptr(), x.data_ptr(), r.data_ptr(), p.data_ptr(), b.numel(),
                                       bb.data_ptr(), ctypes.c_void_p(s.cuda_stream))
    if rc != 0:
        raise lqcd.LqcdError(rc, last_error())
