"""Thin ctypes binding of include/lqcd_slab.h plus the host-side slab bookkeeping.

Time-slab decomposition of the staggered CG: rank r of R owns the
time-slices [r*T, (r+1)*T), T = L3/R even.  Two kinds of code live here, neither with any of the
method's arithmetic:

* index bookkeeping on the canonical layouts of include/lqcd.h (which rows of a global array are a
  rank's, which links are the ``u3_below`` ghost) and its transport between ranks with
  ``torch.distributed`` -- used at set-up time only, covered by world-size-2 gloo tests on CPU;
* argument marshalling for the C-ABI (``Slab``, ``SlabGroup``).  Every step of the hot path --
  hopping terms, halo exchange through peer memory, cross-rank sums, the CG -- runs in the CUDA
  library.  There is no CPU fallback.
"""
from __future__ import annotations

import ctypes
import os
import re

import torch

from . import lqcd as _lqcd
from .lqcd import EVEN, ODD, LqcdError  # noqa: F401

ECOMM = -6
MAX_RANKS = 16
OPT_RECONSTRUCT, OPT_CHECK_EVERY, OPT_TIMEOUT_MS, OPT_GRAPH, OPT_FUSE_SYNC, OPT_ACQUIRE = 0, 1, 2, 3, 4, 5

_HEADER = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "lqcd_slab.h")


def exported_symbols() -> list[str]:
    """Every function include/lqcd_slab.h declares."""
    text = re.sub(r"/\*.*?\*/", "", open(_HEADER).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(lqcd_slab_[a-zA-Z0-9_]+)\s*\(", text)))


# ---------------------------------------------------------------------------- bookkeeping (host)
def slab_extent(dims, nranks: int) -> int:
    """T = L3 / nranks; must be an even integer >= 2 (even slabs keep local parity = global parity)."""
    L3 = int(dims[3])
    if nranks < 1 or nranks > MAX_RANKS or L3 % nranks:
        raise ValueError("L3 = %d cannot be cut into %d slabs" % (L3, nranks))
    T = L3 // nranks
    if T < 2 or T % 2:
        raise ValueError("slab extent T = %d must be even and >= 2" % T)
    return T


def half_slice(dims) -> int:
    """sh: sites of one parity in one time-slice."""
    return int(dims[0]) * int(dims[1]) * int(dims[2]) // 2


def local_dims(dims, nranks: int):
    return (int(dims[0]), int(dims[1]), int(dims[2]), slab_extent(dims, nranks))


def neighbours(rank: int, nranks: int):
    """(rank below, rank above) on the periodic ring of slabs."""
    return (rank - 1) % nranks, (rank + 1) % nranks


def site_range(dims, rank: int, nranks: int):
    """Half-lattice index range [e0, e1) of the rank's slab (the same for both parities and for vectors)."""
    T, sh = slab_extent(dims, nranks), half_slice(dims)
    return rank * T * sh, (rank + 1) * T * sh


def local_vector(v_global: torch.Tensor, dims, rank: int, nranks: int) -> torch.Tensor:
    """Rows of a global staggered vector (3, Vh) that live on the rank's slab: (3, T*sh)."""
    e0, e1 = site_range(dims, rank, nranks)
    return v_global[:, e0:e1].contiguous()


def gather_vector(parts) -> torch.Tensor:
    """Inverse of local_vector over all ranks (parts in rank order)."""
    return torch.cat(list(parts), dim=1).contiguous()


def local_gauge(u_global: torch.Tensor, dims, rank: int, nranks: int) -> torch.Tensor:
    """Canonical gauge field (V, 4, 3, 3) of the local lattice: even sites of the slab, then odd sites."""
    vh = u_global.shape[0] // 2
    e0, e1 = site_range(dims, rank, nranks)
    return torch.cat([u_global[e0:e1], u_global[vh + e0:vh + e1]], dim=0).contiguous()


def u3_top_slice(u_local: torch.Tensor, dims, nranks: int) -> torch.Tensor:
    """U_3 on the LAST time-slice of a local gauge field, (2, sh, 3, 3): what the rank above needs as u3_below."""
    T, sh = slab_extent(dims, nranks), half_slice(dims)
    vh = T * sh
    return torch.stack([u_local[(T - 1) * sh:vh, 3], u_local[vh + (T - 1) * sh:2 * vh, 3]], dim=0).contiguous()


def u3_below_from_global(u_global: torch.Tensor, dims, rank: int, nranks: int) -> torch.Tensor:
    """U_3 on global time-slice t0 - 1 (periodic), (2, sh, 3, 3), cut from a global field."""
    T, sh = slab_extent(dims, nranks), half_slice(dims)
    vh = u_global.shape[0] // 2
    tb = (rank * T - 1) % int(dims[3])
    return torch.stack([u_global[tb * sh:(tb + 1) * sh, 3], u_global[vh + tb * sh:vh + (tb + 1) * sh, 3]], dim=0).contiguous()


def exchange_u3_below(u_local: torch.Tensor, dims, rank: int, nranks: int, group=None) -> torch.Tensor:
    """One process per slab: send the top U_3 slice to the rank above, receive u3_below from the rank
    below (torch.distributed point-to-point; set-up time, not the hot path)."""
    import torch.distributed as dist
    top = u3_top_slice(u_local, dims, nranks)
    if nranks == 1:
        return top
    below, above = neighbours(rank, nranks)
    got = torch.empty_like(top)
    ops = [dist.P2POp(dist.isend, top, above, group=group), dist.P2POp(dist.irecv, got, below, group=group)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    return got


# ---------------------------------------------------------------------------- C-ABI
_bound = False


def _lib():
    global _bound
    L = _lqcd.load_library()
    if not _bound:
        P, I, D, Z = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        PP = ctypes.POINTER(P)
        L.lqcd_slab_create.argtypes = [PP, I, I, I, I, I, I]
        L.lqcd_slab_destroy.argtypes = [P]
        L.lqcd_slab_workspace_bytes.argtypes = [P]
        L.lqcd_slab_workspace_bytes.restype = Z
        L.lqcd_slab_mailbox_bytes.argtypes = [P]
        L.lqcd_slab_mailbox_bytes.restype = Z
        L.lqcd_slab_set_memory.argtypes = [P, P, Z, P, Z, P]
        L.lqcd_slab_connect.argtypes = [P, PP]
        L.lqcd_slab_set_option.argtypes = [P, I, I]
        L.lqcd_slab_load_gauge.argtypes = [P, P, P]
        L.lqcd_slab_dslash.argtypes = [P, I, P, P]
        L.lqcd_slab_apply_MdagM.argtypes = [P, D, P, P]
        L.lqcd_slab_cg_solve.argtypes = [P, D, D, I, P, P, ctypes.POINTER(I), ctypes.POINTER(D)]
        L.lqcd_slab_cg_solve_mixed.argtypes = [P, D, D, I, D, P, P, ctypes.POINTER(I), ctypes.POINTER(I), ctypes.POINTER(D)]
        L.lqcd_slab_cg_solve_mixed_group.argtypes = [PP, I, D, D, I, D, PP, PP, ctypes.POINTER(I), ctypes.POINTER(I),
                                                     ctypes.POINTER(D)]
        L.lqcd_slab_dslash_group.argtypes = [PP, I, I, PP, PP]
        L.lqcd_slab_apply_MdagM_group.argtypes = [PP, I, D, PP, PP]
        L.lqcd_slab_cg_solve_group.argtypes = [PP, I, D, D, I, PP, PP, ctypes.POINTER(I), ctypes.POINTER(D)]
        L.lqcd_slab_ipc_export.argtypes = [P, ctypes.c_char_p, ctypes.POINTER(Z)]
        L.lqcd_slab_ipc_open.argtypes = [P, ctypes.c_char_p, Z, PP]
        L.lqcd_slab_ipc_close.argtypes = [P, P, Z]
        L.lqcd_slab_sync_points.argtypes = [P]
        L.lqcd_slab_sync_points.restype = ctypes.c_longlong
        L.lqcd_slab_kernel_launches.argtypes = [P]
        L.lqcd_slab_kernel_launches.restype = ctypes.c_longlong
        L.lqcd_slab_last_error.argtypes = [P]
        L.lqcd_slab_last_error.restype = ctypes.c_char_p
        _bound = True
    return L


def _aligned(t: torch.Tensor) -> int:
    return (t.data_ptr() + 255) // 256 * 256


class Slab:
    """One lqcd_slab (one rank's time-slab) plus the PyTorch-owned workspace, mailbox and stream."""

    def __init__(self, dims, rank: int, nranks: int, device="cuda:0", stream: torch.cuda.Stream | None = None):
        self._lib = _lib()
        self._s = ctypes.c_void_p()
        self.dims = tuple(int(d) for d in dims)
        self.rank, self.nranks = int(rank), int(nranks)
        rc = self._lib.lqcd_slab_create(ctypes.byref(self._s), *self.dims, self.rank, self.nranks)
        if rc != 0:
            self._s = ctypes.c_void_p()
            raise LqcdError(rc, "lqcd_slab_create%r rank %d/%d failed" % (self.dims, rank, nranks))
        self.T = self.dims[3] // self.nranks
        self.sh = half_slice(self.dims)
        self.vector_shape = (3, self.T * self.sh)
        self.device = torch.device(device)
        if not torch.cuda.is_available():
            raise LqcdError(-4, "no CUDA device (the CUDA path is the only path)")
        wb, mb = self._lib.lqcd_slab_workspace_bytes(self._s), self._lib.lqcd_slab_mailbox_bytes(self._s)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            self.workspace = torch.empty(wb + 256, dtype=torch.uint8, device=self.device)
            self.mailbox = torch.empty(mb + 256, dtype=torch.uint8, device=self.device)
        self.mailbox_ptr = _aligned(self.mailbox)
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        self._check(self._lib.lqcd_slab_set_memory(self._s, ctypes.c_void_p(_aligned(self.workspace)), wb,
                                                   ctypes.c_void_p(self.mailbox_ptr), mb,
                                                   ctypes.c_void_p(self.stream.cuda_stream)))
        self._opened = []

    def _check(self, rc):
        if rc < 0:
            raise LqcdError(rc, self._lib.lqcd_slab_last_error(self._s).decode())
        return rc

    def set_option(self, option: int, value: int):
        self._check(self._lib.lqcd_slab_set_option(self._s, int(option), int(value)))

    def connect(self, peer_mailbox_ptrs):
        arr = (ctypes.c_void_p * self.nranks)(*[ctypes.c_void_p(int(p)) for p in peer_mailbox_ptrs])
        self._check(self._lib.lqcd_slab_connect(self._s, arr))

    def connect_ipc(self, group=None):
        """One process per GPU on one node: all-gather the CUDA IPC handles of the mailboxes and map the
        peers' (torch.distributed is the transport of the 73 bytes per rank; set-up time only).
        Collective and failure-safe: a rank whose export or open fails still takes part in every collective
        of this call, and then EVERY rank raises -- no rank is left waiting for one that has given up."""
        import torch.distributed as dist
        if self.nranks == 1:
            self.connect([self.mailbox_ptr])
            return
        dev = self.device if dist.get_backend(group) == "nccl" else torch.device("cpu")
        failure = ""
        handle = ctypes.create_string_buffer(64)
        off = ctypes.c_size_t()
        try:
            self._check(self._lib.lqcd_slab_ipc_export(self._s, handle, ctypes.byref(off)))
        except Exception as exc:  # noqa: BLE001 - reported to every rank below
            failure = "export: %r" % (exc,)
        mine = torch.tensor(list(handle.raw) + list(int(off.value).to_bytes(8, "little")) + [0 if not failure else 1],
                            dtype=torch.uint8).to(dev)
        everyone = [torch.empty_like(mine) for _ in range(self.nranks)]
        dist.all_gather(everyone, mine, group=group)
        raws = [bytes(t.cpu().tolist()) for t in everyone]
        if not failure and any(r[72] for r in raws):
            failure = "a peer could not export its mailbox"
        ptrs = []
        if not failure:
            try:
                for r, raw in enumerate(raws):
                    if r == self.rank:
                        ptrs.append(self.mailbox_ptr)
                        continue
                    out = ctypes.c_void_p()
                    o = int.from_bytes(raw[64:72], "little")
                    self._check(self._lib.lqcd_slab_ipc_open(self._s, raw[:64], o, ctypes.byref(out)))
                    self._opened.append((out.value, o))
                    ptrs.append(out.value)
                self.connect(ptrs)
                torch.cuda.synchronize(self.device)
            except Exception as exc:  # noqa: BLE001
                failure = "open: %r" % (exc,)
        # every mailbox is zeroed and mapped before anyone's first compute call -- or nobody goes on
        ok = torch.tensor([0 if failure else 1], dtype=torch.int32).to(dev)
        dist.all_reduce(ok, op=dist.ReduceOp.MIN, group=group)
        if int(ok.item()) == 0:
            raise LqcdError(ECOMM, "rank %d: mailboxes not connected (%s)" % (self.rank, failure or "a peer failed"))

    def new_vector(self) -> torch.Tensor:
        return torch.zeros(self.vector_shape, dtype=torch.complex128, device=self.device)

    def load_gauge(self, u_local: torch.Tensor, u3_below: torch.Tensor):
        V = self.dims[0] * self.dims[1] * self.dims[2] * self.T
        assert u_local.dtype == torch.complex128 and u_local.is_contiguous() and tuple(u_local.shape) == (V, 4, 3, 3)
        assert u3_below.dtype == torch.complex128 and u3_below.is_contiguous() and tuple(u3_below.shape) == (2, self.sh, 3, 3)
        assert u_local.device == self.device and u3_below.device == self.device
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        self._check(self._lib.lqcd_slab_load_gauge(self._s, ctypes.c_void_p(u_local.data_ptr()),
                                                   ctypes.c_void_p(u3_below.data_ptr())))
        self.stream.synchronize()   # the inputs may be freed by the caller afterwards

    def _vec(self, t):
        assert t.dtype == torch.complex128 and t.is_contiguous() and tuple(t.shape) == self.vector_shape and t.device == self.device
        return ctypes.c_void_p(t.data_ptr())

    def dslash(self, out_parity: int, vin, vout):
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        self._check(self._lib.lqcd_slab_dslash(self._s, int(out_parity), self._vec(vin), self._vec(vout)))
        return vout

    def apply_MdagM(self, mass: float, vin, vout):
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        self._check(self._lib.lqcd_slab_apply_MdagM(self._s, float(mass), self._vec(vin), self._vec(vout)))
        return vout

    def cg_solve(self, mass: float, tol: float, maxiter: int, b, x):
        it, res = ctypes.c_int(), ctypes.c_double()
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        rc = self._check(self._lib.lqcd_slab_cg_solve(self._s, float(mass), float(tol), int(maxiter), self._vec(b),
                                                      self._vec(x), ctypes.byref(it), ctypes.byref(res)))
        return x, it.value, res.value, rc

    def cg_solve_mixed(self, mass: float, tol: float, maxiter: int, b, x, delta: float = 0.1):
        it, nu, res = ctypes.c_int(), ctypes.c_int(), ctypes.c_double()
        self.stream.wait_stream(torch.cuda.current_stream(self.device))
        rc = self._check(self._lib.lqcd_slab_cg_solve_mixed(self._s, float(mass), float(tol), int(maxiter), float(delta),
                                                            self._vec(b), self._vec(x), ctypes.byref(it), ctypes.byref(nu),
                                                            ctypes.byref(res)))
        return x, it.value, nu.value, res.value, rc

    def sync_points(self) -> int:
        return int(self._lib.lqcd_slab_sync_points(self._s))

    def kernel_launches(self) -> int:
        return int(self._lib.lqcd_slab_kernel_launches(self._s))

    def close(self):
        if getattr(self, "_s", None) and self._s.value:
            self.stream.synchronize()
            for ptr, off in self._opened:
                self._lib.lqcd_slab_ipc_close(self._s, ctypes.c_void_p(ptr), off)
            self._opened = []
            self._lib.lqcd_slab_destroy(self._s)
            self._s = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class SlabGroup:
    """All R slabs of a lattice driven by this process through the *_group calls.  With one device and
    one stream (the default) this runs the complete multi-rank path on a single GPU: the kernels,
    the peer stores and the flags are those of an R-GPU run, and stream order guarantees that no
    kernel ever has to wait for another.  `devices` may instead name R peer-accessible GPUs."""

    def __init__(self, dims, nranks: int, devices=None, recon: int = 18):
        self.dims = tuple(int(d) for d in dims)
        self.nranks = int(nranks)
        slab_extent(self.dims, self.nranks)
        devices = list(devices) if devices is not None else ["cuda:0"] * self.nranks
        assert len(devices) == self.nranks
        same = len({str(torch.device(d)) for d in devices}) == 1
        shared = torch.cuda.Stream(device=torch.device(devices[0])) if same else None
        self.slabs = [Slab(self.dims, r, self.nranks, device=devices[r], stream=shared) for r in range(self.nranks)]
        for s in self.slabs:
            s.set_option(OPT_RECONSTRUCT, recon)
        ptrs = [s.mailbox_ptr for s in self.slabs]
        for s in self.slabs:
            s.connect(ptrs)
        self._lib = self.slabs[0]._lib
        self._arr = (ctypes.c_void_p * self.nranks)(*[s._s.value for s in self.slabs])

    def set_option(self, option: int, value: int):
        for s in self.slabs:
            s.set_option(option, value)

    def load_gauge_from_global(self, u_global: torch.Tensor):
        """u_global: canonical (V, 4, 3, 3) on the host; each slab gets its rows and its u3_below."""
        for s in self.slabs:
            ul = local_gauge(u_global, self.dims, s.rank, self.nranks).to(s.device)
            ub = u3_below_from_global(u_global, self.dims, s.rank, self.nranks).to(s.device)
            s.load_gauge(ul, ub)

    def scatter(self, v_global: torch.Tensor):
        return [local_vector(v_global, self.dims, s.rank, self.nranks).to(s.device) for s in self.slabs]

    def new_vectors(self):
        return [s.new_vector() for s in self.slabs]

    def _ptrs(self, vs):
        return (ctypes.c_void_p * self.nranks)(*[s._vec(v) for s, v in zip(self.slabs, vs)])

    def _pre(self):
        for s in self.slabs:
            s.stream.wait_stream(torch.cuda.current_stream(s.device))

    def _check(self, rc):
        if rc < 0:
            msgs = [s._lib.lqcd_slab_last_error(s._s).decode() for s in self.slabs]
            raise LqcdError(rc, "; ".join(m for m in msgs if m))
        return rc

    def dslash(self, out_parity: int, vin, vout):
        self._pre()
        self._check(self._lib.lqcd_slab_dslash_group(self._arr, self.nranks, int(out_parity), self._ptrs(vin), self._ptrs(vout)))
        return vout

    def apply_MdagM(self, mass: float, vin, vout):
        self._pre()
        self._check(self._lib.lqcd_slab_apply_MdagM_group(self._arr, self.nranks, float(mass), self._ptrs(vin), self._ptrs(vout)))
        return vout

    def cg_solve(self, mass: float, tol: float, maxiter: int, b, x):
        it, res = ctypes.c_int(), ctypes.c_double()
        self._pre()
        rc = self._check(self._lib.lqcd_slab_cg_solve_group(self._arr, self.nranks, float(mass), float(tol), int(maxiter),
                                                            self._ptrs(b), self._ptrs(x), ctypes.byref(it), ctypes.byref(res)))
        return x, it.value, res.value, rc

    def cg_solve_mixed(self, mass: float, tol: float, maxiter: int, b, x, delta: float = 0.1):
        it, nu, res = ctypes.c_int(), ctypes.c_int(), ctypes.c_double()
        self._pre()
        rc = self._check(self._lib.lqcd_slab_cg_solve_mixed_group(self._arr, self.nranks, float(mass), float(tol), int(maxiter),
                                                                  float(delta), self._ptrs(b), self._ptrs(x), ctypes.byref(it),
                                                                  ctypes.byref(nu), ctypes.byref(res)))
        return x, it.value, nu.value, res.value, rc

    def synchronize(self):
        for s in self.slabs:
            s.stream.synchronize()

    def kernel_launches(self) -> int:
        return sum(s.kernel_launches() for s in self.slabs)

    def close(self):
        for s in self.slabs:
            s.close()
