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
