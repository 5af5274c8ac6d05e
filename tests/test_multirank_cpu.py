"""world_size-2 `gloo` test of the N > 1 path on CPU (replicas only -- every
rank solves its own right-hand side, no data-path collective; only timing reductions)."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


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
    from paper_1311_2719_b200 import synth
    from paper_1311_2719_b200.ranks import Ranks
    r = Ranks(backend="gloo")
    seed = r.rhs_seed(131127190 + 1)
    b = synth.source((4, 4, 4, 4), "staggered", seed)
    r.barrier()
    res = dict(rank=r.rank, world=r.world, root=r.is_root, seed=seed, bsum=float(np.abs(b).sum()),
               tmax=r.max(1.0 + rank), wsum=r.sum(10.0 * (rank + 1)),
               thr=r.throughput(10.0 * (rank + 1), 1.0 + rank))
    r.close()
    out.put(res)


def test_two_ranks_gloo_replicas():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(i, 2, port, q)) for i in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=120) for _ in procs), key=lambda d: d["rank"])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g["rank"] for g in got] == [0, 1] and all(g["world"] == 2 for g in got)
    assert got[0]["root"] and not got[1]["root"]
    # independent right-hand sides: rank 0 keeps the BASELINE.json seed, rank 1 a different one
    assert got[0]["seed"] == 131127191 and got[1]["seed"] == 131127191 + 1000
    assert got[0]["bsum"] != got[1]["bsum"]
    # time = max over ranks, work = sum over ranks, whole-job throughput = sum / max on every rank
    for g in got:
        assert g["tmax"] == 2.0 and g["wsum"] == 30.0 and g["thr"] == 15.0


def test_single_rank_needs_no_process_group():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_1311_2719_b200.ranks import Ranks
    r = Ranks(backend="gloo")
    assert r.world == 1 and r.is_root and r.max(3.5) == 3.5 and r.sum(2.0) == 2.0
    assert r.throughput(8.0, 2.0) == 4.0
    r.barrier()
    r.close()


# ------------------------------------------------------------------ bench.py's guarded slab leg: no rank is left behind
def _strong_worker(rank, world, port, fail_on, out):
    """bench.slab_strong_variant with a stand-in Slab that fails on the ranks of `fail_on`: every rank must come back
    with an error dict (none may be left in a collective the other has abandoned)."""
    import argparse
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch
    import bench
    from paper_1311_2719_b200 import slab as sl, synth
    from paper_1311_2719_b200.ranks import Ranks

    class FakeSlab:
        def __init__(self, dims, r, n, device=None):
            if ("create", r) in fail_on:
                raise RuntimeError("no device on rank %d" % r)
            self.rank = r

        def set_option(self, *a):
            pass

        def connect_ipc(self):
            if ("connect", self.rank) in fail_on:
                raise RuntimeError("ipc open failed on rank %d" % self.rank)

        def close(self):
            pass

    sl.Slab = FakeSlab
    r = Ranks(backend="gloo")
    args = argparse.Namespace(recon=18, check_every=8)
    res = bench.slab_strong_variant(args, synth.config(1), r, torch.device("cpu"), 100)
    bad = bench.slab_strong_variant(args, dict(synth.config(1), dims=(4, 4, 4, 6)), r, torch.device("cpu"), 100)
    r.close()
    out.put(dict(rank=rank, res=res, bad=bad))


def _run_strong(fail_on):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_strong_worker, args=(i, 2, port, fail_on, q)) for i in range(2)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=120) for _ in procs), key=lambda d: d["rank"])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    return got


def test_guarded_slab_leg_fails_on_every_rank_when_one_rank_fails():
    for fail_on in ({("create", 1)}, {("create", 0)}, {("connect", 1)}):
        got = _run_strong(fail_on)
        where = "set-up" if ("create", 0) in fail_on or ("create", 1) in fail_on else "connect_ipc"
        for g in got:
            assert set(g["res"]) == {"error"} and g["res"]["error"].startswith(where), g
            assert "cannot be cut" in g["bad"]["error"]          # 6 time-slices in two slabs of three: refused on every rank
        failing = next(r for (_, r) in fail_on)
        assert "rank %d" % failing in got[failing]["res"]["error"] and "a peer failed" in got[1 - failing]["res"]["error"]
