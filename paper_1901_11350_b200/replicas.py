"""Multi-GPU bookkeeping: replicas only.

The hot path has no exchange step on one GPU per lattice, so N GPUs advance N independent lattices (different seeds /
temperatures / images).  This module holds the host logic of that mode -- which replica a rank runs and how the per-rank
device times become one whole-job number -- so that it can be tested on CPU with the gloo backend.  No data-path collective.
"""
from __future__ import annotations

import dataclasses


def replica_workload(w, rank: int):
    """The workload of replica `rank`: same lattice and Hamiltonian, its own noise / initial-state seed."""
    return dataclasses.replace(w, seed=int(w.seed) + 1000003 * int(rank), name=f"{w.name}#r{rank}" if rank else w.name)


def max_over_ranks(ms: float, device=None) -> float:
    """Slowest rank's device time (ms): one all-reduce(MAX) of a scalar; identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(spins_per_rank: int, iterations: int, ms_max: float, world: int) -> float:
    """spin-updates/s of the whole job: all ranks' updates over the slowest rank's time (weak scaling)."""
    return world * spins_per_rank * iterations / (ms_max * 1e-3)
