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


# ---------------------------------------------------------------------------------------------------------------------
# Fused halo exchange between processes (slab.py: fused_links, fused_step_ops; include/spinllg.h llg_slab_step_fused): the kernel writes
# its boundary planes into the neighbours' arrays, mapped through CUDA IPC, and flags in device memory keep the order of the steps.  The
# device side is covered on the GPU with all slabs in one process; here: who maps whose export, which flag each rank writes, and that the
# wait / step / signal sequence lets no rank read a ghost layer before it was written or write into an array that is still being read.
def _links_worker(rank, world, port, out, periodic, n_planes):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        plan = S.HaloPlan.make(rank, world, n_planes, periodic, 2)
        mine = {"rank": rank, "count": plan.count, "arrays": ((b"cur%d" % rank, 0), (b"next%d" % rank, 64)), "flags": (b"flags%d" % rank, 16 * rank)}
        infos = [None] * world
        dist.all_gather_object(infos, mine)
        links = S.fused_links(plan, infos)
        ok = len(links) == 2
        for side in (0, 1):
            peer = plan.neighbour(side)
            if peer is None:
                ok &= links[side] is None
                continue
            ln = links[side]
            ok &= ln.rank == peer and ln.count == S.partition(n_planes, world)[peer][1] and ln.signal_index == 1 - side
            ok &= ln.arrays == ((b"cur%d" % peer, 0), (b"next%d" % peer, 64)) and ln.flags == (b"flags%d" % peer, 16 * peer)
        res = [None] * world
        dist.all_gather_object(res, bool(ok))
        if rank == 0:
            out.put(res)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
@pytest.mark.parametrize("world,periodic,n_planes", [(2, True, 17), (2, False, 16), (3, True, 25)])
def test_fused_links_gloo(world, periodic, n_planes):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_links_worker, args=(r, world, port, out, periodic, n_planes)) for r in range(world)]
    for p in procs:
        p.start()
    res = out.get(timeout=150)
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    assert res == [True] * world


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True), (4, False), (5, True)])
def test_fused_step_protocol_orders_reads_and_writes(world, periodic):
    """Every rank's stream executes fused_step_ops in order; a random scheduler interleaves the ranks (a step is split into its reads and
    its writes).  Arrays are modelled by version numbers: step k reads the arrays of parity k - 1 -- own planes and both ghost layers
    must hold version k - 1 -- and writes version k into its own array of parity k and into the neighbours' ghost layers of that array."""
    import random
    rng = random.Random(1234 + world)
    steps = 12
    plans = [S.HaloPlan.make(r, world, 8 * world, periodic, 2) for r in range(world)]
    links = [S.fused_links(p, [{"rank": q, "count": 8, "arrays": ((b"c", 0), (b"n", 0)), "flags": (b"f", 0)} for q in range(world)]) for p in plans]
    sides = [[s for s in (0, 1) if links[r][s] is not None] for r in range(world)]
    ops = []
    for r in range(world):
        seq = []
        for k in range(1, steps + 1):
            for op in S.fused_step_ops(k, sides[r]):
                seq += [("read", k), ("write", k)] if op[0] == "step" else [op]
        ops.append(seq)
    flags = [[0, 0] for _ in range(world)]
    own = [[0, 0] for _ in range(world)]                      # own[r][parity]: version of the own planes (both arrays hold the start: 0)
    ghost = [[[0, 0], [0, 0]] for _ in range(world)]          # ghost[r][parity][side]
    reading = [None] * world                                  # parity a rank is reading between its "read" and its "write"
    pc = [0] * world
    while any(pc[r] < len(ops[r]) for r in range(world)):
        ready = [r for r in range(world) if pc[r] < len(ops[r]) and not (ops[r][pc[r]][0] == "wait" and flags[r][ops[r][pc[r]][1]] < ops[r][pc[r]][2])]
        assert ready, "deadlock"
        r = rng.choice(ready)
        op = ops[r][pc[r]]
        pc[r] += 1
        if op[0] == "read":
            k = op[1]
            q = (k - 1) % 2
            assert own[r][q] == k - 1 or k == 1
            for s in sides[r]:
                assert ghost[r][q][s] == k - 1 or k == 1, (r, k, s, ghost[r][q])
            reading[r] = q
        elif op[0] == "write":
            k = op[1]
            q = k % 2
            own[r][q] = k
            reading[r] = None
            for s in sides[r]:
                p = links[r][s].rank
                assert reading[p] != q, f"rank {r} step {k} writes into the array rank {p} is reading"
                ghost[p][q][1 - s] = k                        # this rank is on side 1 - s of that neighbour
        elif op[0] == "signal":
            ln = links[r][op[1]]
            flags[ln.rank][ln.signal_index] = op[2]
    assert all(own[r][steps % 2] == steps for r in range(world))
