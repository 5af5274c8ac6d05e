"""One process per GPU: the rank plumbing bench.py and the multi-rank drivers share.

The path of arXiv 1311.2719 runs on one GPU (BASELINE.json); with N > 1 processes every rank
owns independent right-hand sides on the same gauge field (the replicas mode of DESIGN.md section 8;
the time-slab decomposition of one system lives in slab.py and include/lqcd_slab.h):
no data-path collective, only the timing reductions below.  `torch.distributed` is the
transport: NCCL on GPUs, gloo in the CPU tests (world_size 2, 127.0.0.1).

Nothing here touches the method's arithmetic.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


class Ranks:
    """RANK / LOCAL_RANK / WORLD_SIZE from the environment (torchrun's contract) plus the three
    reductions a benchmark needs: barrier, max over ranks (time), sum over ranks (work)."""

    def __init__(self, backend: str | None = None, device: torch.device | None = None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device if device is not None else torch.device("cpu")
        self.backend = backend or ("nccl" if self.device.type == "cuda" else "gloo")
        self._own_group = False
        if self.world > 1 and not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            kw = {}
            if self.backend == "nccl":
                kw["device_id"] = self.device
            dist.init_process_group(self.backend, rank=self.rank, world_size=self.world, **kw)
            self._own_group = True

    # -- reductions -------------------------------------------------------------------------
    def _reduce(self, x: float, op) -> float:
        if self.world == 1:
            return float(x)
        t = torch.tensor([x], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=op)
        return float(t.item())

    def max(self, x: float) -> float:
        return self._reduce(x, dist.ReduceOp.MAX)

    def sum(self, x: float) -> float:
        return self._reduce(x, dist.ReduceOp.SUM)

    def barrier(self) -> None:
        if self.world > 1:
            dist.barrier()
        if self.device.type == "cuda":
            torch.cuda.synchronize(self.device)

    # -- work split -------------------------------------------------------------------------
    def rhs_seed(self, base_seed: int) -> int:
        """Seed of this rank's right-hand side: rank 0 solves the BASELINE.json source itself."""
        return int(base_seed) + 1000 * self.rank

    def throughput(self, units_this_rank: float, seconds_this_rank: float) -> float:
        """Whole-job throughput: the units all ranks processed / the slowest rank's time."""
        return self.sum(units_this_rank) / self.max(seconds_this_rank)

    @property
    def is_root(self) -> bool:
        return self.rank == 0

    def close(self) -> None:
        if self._own_group and dist.is_initialized():
            dist.destroy_process_group()
            self._own_group = False
