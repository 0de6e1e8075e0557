"""topological_charge_noalloc (include/spinllg.h): the entry point for callers that must not allocate.  Its per-block partial sums live in
a fixed file-scope device array shared by every call, so the checks are: the same value as topological_charge (same kernels, same order
of additions: the tolerance is that of the other topological-charge tests and the values are in fact identical), on calls in a row whose
systems differ in size (a smaller system after a larger one must not see the larger one's partial sums), and the stated size limit.
Collected last on purpose (the suite runs with pytest -x)."""
import dataclasses

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-10      # the absolute tolerance test_topological_charge_parity uses for an integer charge


@pytest.fixture(scope="module")
def P():
    import paper_1901_11350_b200 as P
    return P


def _system(P, cfg, cells, per):
    w = dataclasses.replace(W.CONFIGS[cfg]().resized(cells, 4), periodic=per)
    return w, P.SpinSystem.from_workload(w)


def test_noalloc_topological_charge_matches_the_allocating_path_on_calls_in_a_row(P):
    import torch
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    wa, a = _system(P, 1, (96, 70, 3), (1, 1, 0))        # 20160 cells: 79 blocks of partial sums
    wb, b = _system(P, 1, (20, 11, 1), (0, 1, 0))        # 220 cells: one block, run right after the larger system
    calls = []
    for sysm, w, spins in ((a, wa, W.skyrmion_spins(wa, 9.0)), (b, wb, wb.initial_spins()), (a, wa, wa.initial_spins()),
                           (a, wa, None), (b, wb, W.skyrmion_spins(wb, 4.0))):
        if spins is None:                                  # a configuration reached by time stepping, not set from the host
            sysm.llg_iterate(4)
        else:
            sysm.spins_set(spins)
        want = sysm.topological_charge()
        sysm.topological_charge_noalloc(out.data_ptr())
        sysm.spin_synchronize()
        got = float(out.cpu()[0])
        calls.append((want, got))
        assert abs(got - want) <= TOL, calls
    # two calls in a row on one system without anything in between
    a.topological_charge_noalloc(out.data_ptr())
    a.topological_charge_noalloc(out.data_ptr())
    a.spin_synchronize()
    assert abs(float(out.cpu()[0]) - a.topological_charge()) <= TOL
    # the periodic skyrmion films carry an integer charge per plane: the values are not trivially zero
    assert abs(calls[0][0] + 3.0) <= TOL, calls


def test_noalloc_topological_charge_limits(P):
    import torch
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    # the plan must exist already (building it allocates)
    _, fresh = _system(P, 1, (16, 16, 1), (1, 1, 0))
    fresh.llg_configure(1e-3, 0.2)                        # marks the plan as out of date
    with pytest.raises(P.SpinError, match="plan"):
        fresh.topological_charge_noalloc(out.data_ptr())
    fresh.topological_charge()
    fresh.topological_charge_noalloc(out.data_ptr())
    fresh.spin_synchronize()
    assert abs(float(out.cpu()[0]) - fresh.topological_charge()) <= TOL
    # one basis atom only, like topological_charge
    two = P.SpinSystem.from_workload(W.config4().resized((8, 8, 1), 1))
    with pytest.raises(P.SpinError):
        two.topological_charge_noalloc(out.data_ptr())
    # more cells than the fixed array covers (16384 blocks of 256 cells): a clear error, nothing launched
    big = P.SpinSystem(np.eye(3), [[0, 0, 0]], (2049, 2048, 1), (1, 1, 0), 1.0)
    with pytest.raises(P.SpinError, match="exceed"):
        big.topological_charge_noalloc(out.data_ptr())
    big.close()
    with pytest.raises(P.SpinError):
        fresh.topological_charge_noalloc(0)
