"""World-size-2 CPU tests (gloo) of the N>1 path: band sharding with NO data-path collective.

DESIGN.md "Multi-GPU": bands are independent in project (eq. (25) carries the band index k freely,
PAPER.md:246) and in add (step (3)), so rank r owns ``band_range(nbands, r, N)`` and the
only communication is bench.py's timing protocol.  There is one GPU at most in this run, so the
per-rank compute of these tests is the CPU oracle (tests may use it); what is under test is the host
logic: the shard bookkeeping, that sharded results concatenate to the unsharded result bit for bit,
and the barrier / max-over-ranks reduction bench.py reports.
"""
import os
import socket

import numpy as np
import pytest

from paper_1905_00480_b200 import sharding, workloads


def test_band_range_partitions_every_band_once():
    for nbands in (0, 1, 3, 16, 31, 64):
        for world in (1, 2, 3, 4, 8):
            seen = []
            sizes = []
            for r in range(world):
                lo, hi = sharding.band_range(nbands, r, world)
                assert 0 <= lo <= hi <= nbands
                seen += list(range(lo, hi))
                sizes.append(hi - lo)
                for b in range(lo, hi):
                    assert sharding.band_owner(b, nbands, world) == r
            assert seen == list(range(nbands))              # contiguous, ascending, exactly once
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.band_range(4, 2, 2)
    with pytest.raises(ValueError):
        sharding.band_owner(4, 4, 2)


def test_max_over_ranks_is_identity_without_a_process_group():
    assert sharding.max_over_ranks([1.5, 2.0]) == [1.5, 2.0]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, k, q):
    import torch
    import torch.distributed as dist

    import oracle

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.make(k, size="small")
        wide = np.complex128 if w.is_complex else np.float64
        nb = w.nbands
        lo, hi = sharding.band_range(nb, rank, world)
        geo = (w.ng, w.h, w.periodic, w.kfrac, w.pos, w.sigma, w.numax)
        # every rank regenerates only ITS bands (workloads draws each band from its own seed)
        psi_loc = w.psi(range(lo, hi)).astype(wide)
        c_loc = oracle.project(*geo, psi_loc, w.rcut_sigma)                       # [natoms][hi-lo][nsho]
        psi_new = oracle.add(*geo, c_loc, psi_loc, w.rcut_sigma)                  # psi += A c on the shard
        dist.barrier()
        c_all = sharding.gather_band_slabs(torch.from_numpy(c_loc), nb, band_axis=1).numpy()
        psi_all = sharding.gather_band_slabs(torch.from_numpy(psi_new), nb, band_axis=0).numpy()
        # bench.py's timing reduction: the slowest rank decides
        t = sharding.max_over_ranks([1.0 + rank, 10.0 - rank])
        if rank == 0:
            psi_full = w.psi().astype(wide)
            c_ref = oracle.project(*geo, psi_full, w.rcut_sigma)
            psi_ref = oracle.add(*geo, c_ref, psi_full, w.rcut_sigma)
            q.put({"c_equal": bool(np.array_equal(c_all, c_ref)), "psi_equal": bool(np.array_equal(psi_all, psi_ref)),
                   "shape": tuple(c_all.shape), "t": t, "nb": nb})
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("k", [2, 5])
def test_band_sharded_project_add_equals_unsharded_world2(k):
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    world = 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, k, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=300)
        assert p.exitcode == 0, "rank failed (exit code %s)" % p.exitcode
    res = q.get()
    assert res["nb"] == 3                                    # odd band count: ranks own 2 and 1 bands
    assert res["c_equal"], "band-sharded projection differs from the unsharded one"
    assert res["psi_equal"], "band-sharded add-back differs from the unsharded one"
    assert res["t"] == [2.0, 10.0]                           # max over ranks of [1+r, 10-r]
