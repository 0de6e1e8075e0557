"""N > 1 path on CPU: replicas only, world_size 2 over gloo.  Covers the rank -> replica mapping and the
max-over-ranks timing reduction that bench.py uses; the data path itself has no collective."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as W
from paper_1901_11350_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = replicas.replica_workload(W.config1(), rank)
        ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
        ms_max = replicas.max_over_ranks(ms)
        seeds = [None] * world
        dist.all_gather_object(seeds, int(w.seed))
        first = w.initial_spins()[0].tolist()
        firsts = [None] * world
        dist.all_gather_object(firsts, first)
        if rank == 0:
            out.put({"ms_max": ms_max, "seeds": seeds, "firsts": firsts,
                     "rate": replicas.whole_job_rate(w.n_spins, 100, ms_max, world)})
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_replicas_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=90)
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    assert res["ms_max"] == 15.0                                  # the slowest rank sets the time
    assert res["seeds"][0] == W.config1().seed and res["seeds"][1] != res["seeds"][0]
    assert res["firsts"][0] != res["firsts"][1]                   # replicas start from different configurations
    assert res["rate"] == pytest.approx(2 * 1024 * 100 / 15e-3)   # whole-job aggregate over the slowest rank's time


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.replica_workload(W.config3(), 0).seed == W.config3().seed


# ---------------------------------------------------------------------------------------------------------------------
# Slab decomposition along c (paper_1901_11350_b200/slab.py): the halo bookkeeping on CPU.  Each rank holds a numpy slab with ghost
# layers; after `exchange` over gloo every ghost plane must be the plane of the global lattice it stands for (periodic wrap included),
# and ghost layers at open ends must be left alone.
from paper_1901_11350_b200 import slab as S


def test_partition_and_halo_plan():
    assert S.partition(128, 4) == [(0, 32), (32, 32), (64, 32), (96, 32)]
    assert S.partition(10, 3) == [(0, 4), (4, 3), (7, 3)]
    with pytest.raises(ValueError):
        S.partition(2, 3)
    for world in (1, 2, 3, 5):
        for periodic in (False, True):
            plans = [S.HaloPlan.make(r, world, 23, periodic, 2) for r in range(world)]
            assert sum(p.count for p in plans) == 23 and plans[0].first == 0
            for p in plans:
                for side in (0, 1):
                    q = p.neighbour(side)
                    if q is None:
                        assert not periodic and ((side == 0 and p.rank == 0) or (side == 1 and p.rank == world - 1))
                        continue
                    # what I receive on `side` is what that neighbour sends towards the opposite side
                    want = [z % 23 for z in p.ghost_planes(side)]
                    assert want == list(plans[q].own_planes(1 - side)), (world, periodic, p.rank, side)
                    assert plans[q].neighbour(1 - side) == p.rank
    with pytest.raises(ValueError):
        S.HaloPlan.make(0, 8, 8, True, 2)            # slabs of one plane cannot serve a reach of two


def _slab_worker(rank, world, port, out, periodic, reach, n_planes):
    import numpy as np
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        plane = 7
        glob = np.arange(n_planes * plane, dtype=np.float64).reshape(n_planes, plane) + 0.5
        plan = S.HaloPlan.make(rank, world, n_planes, periodic, reach)
        local = np.full((plan.count + 2 * reach, plane), np.nan)
        local[reach:reach + plan.count] = glob[plan.first:plan.first + plan.count]

        def get(side, buf):
            lo = reach if side == 0 else plan.count
            buf.copy_(torch.from_numpy(local[lo:lo + reach].reshape(-1).copy()))

        def put(side, buf):
            lo = 0 if side == 0 else reach + plan.count
            local[lo:lo + reach] = buf.numpy().reshape(reach, plane)

        send = [torch.zeros(reach * plane, dtype=torch.float64) for _ in range(2)]
        recv = [torch.zeros(reach * plane, dtype=torch.float64) for _ in range(2)]
        for _ in range(2):                      # twice: tags and ordering must hold for back-to-back exchanges too
            S.exchange(plan, get, put, send, recv, S.DistTransport(dist))
        ok = True
        for side in (0, 1):
            lo = 0 if side == 0 else reach + plan.count
            ghost = local[lo:lo + reach]
            if plan.neighbour(side) is None:
                ok &= bool(np.isnan(ghost).all())
            else:
                ok &= bool(np.array_equal(ghost, glob[[z % n_planes for z in plan.ghost_planes(side)]]))
        ok &= bool(np.array_equal(local[reach:reach + plan.count], glob[plan.first:plan.first + plan.count]))
        res = [None] * world
        dist.all_gather_object(res, ok)
        if rank == 0:
            out.put(res)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
@pytest.mark.parametrize("world,periodic,reach,n_planes", [(2, True, 1, 8), (2, False, 2, 9), (2, True, 2, 5), (3, True, 1, 10)])
def test_halo_exchange_gloo(world, periodic, reach, n_planes):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, out, periodic, reach, n_planes)) for r in range(world)]
    for p in procs:
        p.start()
    res = out.get(timeout=150)
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    assert res == [True] * world
