"""Slab decomposition of one lattice along c over several GPUs.

Each rank holds a slab of consecutive planes; before every sweep its ghost layers along c receive the neighbours' boundary planes
(twice per Depondt step: n before the predictor, n^p before the corrector).  The kernels, the ghost-aware plan and the halo planes as
contiguous device chunks are the C library's (include/spinllg.h "slab decomposition"); this module holds the HOST logic:

  * `partition`        which planes a rank owns (balanced, contiguous);
  * `HaloPlan`         who a rank's neighbours are (periodic ring or open chain) and which of its planes go where;
  * `exchange`         one halo exchange of one array over a transport (`DistTransport`: torch.distributed point-to-point, NCCL between
                       GPUs, gloo in the CPU tests);
  * `SlabDriver`       one rank's step: boundary bricks first, their halos travel on a second stream while the interior bricks run;
  * `LocalGroup`       all slabs in one process on one device (device copies as transport): the 1-GPU emulation of N ranks;
  * one-pass mode      (3-D lattices of one basis atom, Depondt): the plane-marching kernel steps a slab in one pass, ONE exchange of
                       depth 2 x reach per step (`llg_slab_step`);
  * fused exchange     that kernel writes its boundary planes straight into the neighbours' ghost layers (`llg_slab_step_fused`):
                       `LocalGroup(fused=True)` in one process, `SlabDriver.setup_fused` / `iterate_fused` between processes (CUDA IPC
                       mappings, order kept by flags in device memory: `fused_links`, `fused_step_ops`).

Only argument marshalling and ordering happen here; every arithmetic step of the path runs in the library's kernels.  The paper has no
counterpart (MPI appears only as a remark on scripting).
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence, Tuple


def partition(n_planes: int, world: int) -> List[Tuple[int, int]]:
    """[(first plane, plane count)] per rank: contiguous, sizes differ by at most one, larger slabs first."""
    if world < 1 or n_planes < world:
        raise ValueError(f"cannot cut {n_planes} planes into {world} slabs")
    base, extra = divmod(n_planes, world)
    out, first = [], 0
    for r in range(world):
        cnt = base + (1 if r < extra else 0)
        out.append((first, cnt))
        first += cnt
    return out


@dataclasses.dataclass(frozen=True)
class HaloPlan:
    """Neighbours and plane ranges of one rank.  `reach` = ghost width along c (the Hamiltonian's largest |translation| along c)."""
    rank: int
    world: int
    first: int            # first global plane of the slab
    count: int            # planes in the slab
    n_planes: int         # planes of the whole lattice
    periodic: bool
    reach: int

    @staticmethod
    def make(rank: int, world: int, n_planes: int, periodic: bool, reach: int) -> "HaloPlan":
        first, count = partition(n_planes, world)[rank]
        if reach > count:
            raise ValueError(f"rank {rank}: slab of {count} planes is thinner than the reach {reach}")
        return HaloPlan(rank, world, first, count, n_planes, bool(periodic), int(reach))

    # neighbour towards lower / higher c, or None at an open end
    @property
    def lower(self) -> Optional[int]:
        if self.rank > 0:
            return self.rank - 1
        return self.world - 1 if self.periodic else None

    @property
    def upper(self) -> Optional[int]:
        if self.rank < self.world - 1:
            return self.rank + 1
        return 0 if self.periodic else None

    def neighbour(self, side: int) -> Optional[int]:
        return self.lower if side == 0 else self.upper

    def own_planes(self, side: int) -> range:
        """global planes this rank SENDS towards `side` (its outermost `reach` planes on that side)"""
        return range(self.first, self.first + self.reach) if side == 0 else range(self.first + self.count - self.reach, self.first + self.count)

    def ghost_planes(self, side: int) -> range:
        """global planes (modulo the lattice when periodic) this rank RECEIVES into its ghost layer on `side`"""
        lo = self.first - self.reach if side == 0 else self.first + self.count
        return range(lo, lo + self.reach)


class DistTransport:
    """Halo messages over torch.distributed point-to-point calls (NCCL between GPUs; gloo in the CPU tests)."""

    def __init__(self, dist, group=None):
        self.dist, self.group = dist, group

    def sendrecv(self, plan: HaloPlan, send: Sequence, recv: Sequence):
        """send[side] / recv[side]: tensors (or None where there is no neighbour).  The message towards `side` is what the neighbour on
        that side puts into ITS opposite ghost layer.  All four operations are posted before any is waited for (no ordering deadlock);
        tag = the side the message travels towards, so the two messages between a pair of ranks (world = 2, periodic) stay apart."""
        ops = []
        for side in (0, 1):                      # sends in the order low, high ...
            peer = plan.neighbour(side)
            if peer is not None and peer != plan.rank:
                ops.append(self.dist.P2POp(self.dist.isend, send[side], peer, self.group, tag=side))
        for side in (1, 0):                      # ... receives in the order high, low: with ONE peer on both sides (two ranks on a ring) the
            peer = plan.neighbour(side)          # peer's first send (its low planes) is this rank's high ghost layer -- NCCL matches by order,
            if peer is not None and peer != plan.rank:      # gloo by tag
                ops.append(self.dist.P2POp(self.dist.irecv, recv[side], peer, self.group, tag=1 - side))
        if plan.world == 1 and plan.periodic:        # a ring of one: the slab is its own neighbour
            recv[0].copy_(send[1]); recv[1].copy_(send[0])
        for w in (self.dist.batch_isend_irecv(ops) if ops else []):
            w.wait()


class StagedTransport(DistTransport):
    """The same messages staged through host memory: for backends that move host tensors only (gloo) -- tests, or a node without NCCL."""

    def sendrecv(self, plan: HaloPlan, send: Sequence, recv: Sequence):
        hs = [None if t is None else t.cpu() for t in send]
        hr = [None if t is None else t.cpu() for t in recv]
        super().sendrecv(plan, hs, hr)
        for d, h in zip(recv, hr):
            if d is not None:
                d.copy_(h)


def exchange(plan: HaloPlan, get, put, send_buf, recv_buf, transport) -> None:
    """One halo exchange of one array: get(side, buffer) fills buffer with the own boundary planes of `side`; the transport moves
    send_buf[side] to the neighbour on that side, whose message arrives in recv_buf[side]; put(side, buffer) writes the ghost planes."""
    for side in (0, 1):
        if plan.neighbour(side) is not None:
            get(side, send_buf[side])
    transport.sendrecv(plan, send_buf, recv_buf)
    for side in (0, 1):
        if plan.neighbour(side) is not None:
            put(side, recv_buf[side])


@dataclasses.dataclass(frozen=True)
class FusedLink:
    """What one rank needs to know about the neighbour on one side for the fused exchange between processes (llg_slab_step_fused)."""
    rank: int                 # the neighbour
    count: int                # planes of its slab
    arrays: tuple             # exports (handle, offset) of its (current, next) configuration arrays AT SET-UP; they swap every step
    flags: tuple              # export of its two step flags
    signal_index: int         # which of ITS flags this rank writes: 1 if this rank is its upper neighbour, 0 if its lower


def fused_links(plan: HaloPlan, infos: Sequence[dict]) -> List[Optional[FusedLink]]:
    """links[side] from the gathered per-rank records {rank, count, arrays, flags}.  The lower neighbour (side 0) sees this rank as ITS
    upper neighbour and keeps that neighbour's progress in its flag [1]; the upper neighbour (side 1) in its flag [0].  On a ring of two
    both sides are the same peer: this rank writes both of its flags and waits on both of its own."""
    by_rank = {int(r["rank"]): r for r in infos}
    links: List[Optional[FusedLink]] = []
    for side in (0, 1):
        peer = plan.neighbour(side)
        if peer is None or peer == plan.rank:
            links.append(None)
            continue
        r = by_rank[peer]
        links.append(FusedLink(peer, int(r["count"]), tuple(r["arrays"]), tuple(r["flags"]), 1 - side))
    return links


def fused_step_ops(step: int, sides: Sequence[int]) -> List[tuple]:
    """The stream-ordered operations of fused step number `step` (1, 2, ...) of one rank with neighbours on `sides`: wait until every
    neighbour has finished step - 1 (it wrote this rank's ghost layers and read the arrays this step writes into), step, tell them."""
    return [("wait", side, step - 1) for side in sides] + [("step", step)] + [("signal", side, step) for side in sides]


class SlabDriver:
    """One rank's slab of a workload and its time stepping.

        drv = SlabDriver(P, torch, workload, rank, world, transport)      # builds the local system on the current device
        drv.iterate(n)                                                      # n steps, halos exchanged twice per step
        drv.spins()                                                         # this rank's spins (boundary order of the slab)

    A stage (predictor or corrector) runs in three phases so that N slabs of one process can be driven in lockstep too:
      begin_stage   sweep the brick layers the neighbours need, copy their planes into the send buffers on a second stream, launch the
                    interior layers on the system's stream (they run while the halos travel)
      transport     move send[side] to the neighbour on that side (DistTransport: inside iterate; LocalGroup: between the phases)
      end_stage     write the received planes into the ghost layers; the system's stream waits for that before its next sweep
    """

    def __init__(self, P, torch, w, rank: int, world: int, transport=None, stream=None, options=()):
        self.P, self.torch = P, torch
        na, nb_, nc = (int(x) for x in w.n_cells)
        first, count = partition(nc, world)[rank]
        lw = dataclasses.replace(w, n_cells=(na, nb_, count))
        self.stream = stream if stream is not None else torch.cuda.Stream()
        self.copy_stream = torch.cuda.Stream()
        self.sys = P.SpinSystem.from_workload(lw, stream=self.stream.cuda_stream)
        for name, value in dict(options).items():             # execution options (spin_set_option), the same on every rank
            self.sys.spin_set_option(name, int(value))
        self.sys.spin_set_slab(True, first, nc, int(w.periodic[2]))
        per_plane = self.sys.N // count
        self.sys.spins_set(w.initial_spins().reshape(nc, per_plane, 3)[first:first + count].reshape(-1, 3))      # boundary order: planes are contiguous
        nd, reach = self.sys.spin_halo_doubles()
        # one-pass marching kernel (3-D lattices of one basis atom, Depondt): the slab recomputes the predictor of its neighbours' boundary
        # planes, so a step needs ONE exchange (of the new configuration, ghost depth 2 x reach) instead of two
        self.one_pass = "march" in self.sys.spin_kernel_info()
        self.plan = HaloPlan.make(rank, world, nc, bool(w.periodic[2]), reach)
        self.transport = transport
        dev = torch.device("cuda", torch.cuda.current_device())
        self.send = [torch.zeros(nd, dtype=torch.float64, device=dev) for _ in range(2)]
        self.recv = [torch.zeros(nd, dtype=torch.float64, device=dev) for _ in range(2)]
        self.sent = torch.cuda.Event()
        self.halo_bytes_per_exchange = 8 * nd * sum(1 for side in (0, 1) if self.plan.neighbour(side) is not None)

    # ---- the three phases of one halo exchange of `array` (0 n, 1 n^p, 2 next n)
    def post(self, array: int) -> None:
        """own boundary planes -> send buffers, on the copy stream, after everything enqueued so far on the system's stream"""
        ev = self.torch.cuda.Event()
        ev.record(self.stream)
        self.copy_stream.wait_event(ev)
        for side in (0, 1):
            if self.plan.neighbour(side) is not None:
                self.sys.spin_halo_get(array, side, self.send[side].data_ptr(), self.copy_stream.cuda_stream)
        self.sent.record(self.copy_stream)

    def deliver(self, array: int) -> None:
        """received planes -> ghost layers; the system's stream waits for them"""
        for side in (0, 1):
            if self.plan.neighbour(side) is not None:
                self.sys.spin_halo_put(array, side, self.recv[side].data_ptr(), self.copy_stream.cuda_stream)
        done = self.torch.cuda.Event()
        done.record(self.copy_stream)
        self.stream.wait_event(done)

    def begin_stage(self, stage: int, array: int) -> None:
        self.sys.llg_slab_sweep(stage, 1)
        self.post(array)
        self.sys.llg_slab_sweep(stage, 2)

    def begin_step(self) -> None:
        """one-pass mode: the chunks of planes the neighbours need, their halo copies on the second stream, the chunks in between"""
        self.sys.llg_slab_step(1)
        self.post(2)
        self.sys.llg_slab_step(2)

    def stages(self):
        """(begin, array) of every exchange of one step"""
        if self.one_pass:
            return [(self.begin_step, 2)]
        return [(lambda: self.begin_stage(0, 1), 1), (lambda: self.begin_stage(1, 2), 2)]

    def _transport(self) -> None:
        with self.torch.cuda.stream(self.copy_stream):
            self.transport.sendrecv(self.plan, self.send, self.recv)

    def exchange_initial(self) -> None:
        self.post(0); self._transport(); self.deliver(0)

    def iterate(self, n_steps: int) -> None:
        """n steps of this rank (every rank calls it with the same n)"""
        if not getattr(self, "_primed", False):              # ghosts of the configuration the run starts from
            self.exchange_initial()
            self._primed = True
        for _ in range(int(n_steps)):
            for begin, array in self.stages():          # two-sweep mode: predictor + halos of n^p, corrector + halos of the next n
                begin(); self._transport(); self.deliver(array)
            self.sys.llg_slab_advance()

    # ---- fused exchange between processes: neighbours' arrays mapped through CUDA IPC, order kept by flags in device memory
    def setup_fused(self, dist, group=None, order: str = "flags") -> None:
        """Collective over the group, once: exchange the IPC exports and map the neighbours' arrays and flags.  Needs the one-pass kernel on
        every rank, one rank per GPU with peer access between neighbours, and ghost layers that are current (iterate primes them).
        Every kernel that runs while a wait polls has run before: the flag kernels in spin_slab_flags, the step's kernels in the first
        step, whose waits (for step 0) pass at once -- a kernel's first launch may load code, which waits for the device."""
        if not self.one_pass:
            raise ValueError("the fused exchange needs the one-pass kernel (spin_kernel_info: %s)" % self.sys.spin_kernel_info())
        if getattr(self, "_links", None) is not None:
            return                            # set up already: the mappings and the step count of the flags stay
        if not getattr(self, "_primed", False):
            self.exchange_initial()
            self._primed = True
        self.synchronize()
        cur, nxt = self.sys.spin_slab_arrays()
        self._cur0 = cur                      # which of the two arrays was the current one at set-up: the same on every rank (lockstep)
        self._flags = self.sys.spin_slab_flags()
        mine = {"rank": self.plan.rank, "count": self.plan.count, "arrays": (self.P.spin_ipc_export(cur), self.P.spin_ipc_export(nxt)),
                "flags": self.P.spin_ipc_export(self._flags)}
        infos = [None] * self.plan.world
        dist.all_gather_object(infos, mine, group=group)
        self._links = fused_links(self.plan, infos)
        self._peer = []                       # per side: [address of its current-at-set-up array, of its other array, of the flag this rank writes]
        opened = {}                           # (a ring of two: one peer on both sides, each export mapped once)
        for link in self._links:
            if link is None:
                self._peer.append(None)
                continue
            addr = []
            for handle, off in (link.arrays[0], link.arrays[1], link.flags):
                key = (link.rank, handle)
                if key not in opened:
                    opened[key] = self.P.spin_ipc_open(handle, 0)
                addr.append(opened[key] + off)
            self._peer.append([addr[0], addr[1], addr[2] + 8 * link.signal_index])
        self._opened = list(opened.values())
        self._fused_step = 0
        # order = "host": a host barrier after every step instead of the flags (slow; for ranks that share a GPU, where a polling kernel
        # of one rank would keep the other rank's kernels from running)
        self._order, self._dist, self._group = order, dist, group
        dist.barrier(group=group)             # nobody steps before every mapping exists

    def close_fused(self) -> None:
        """unmap the neighbours' arrays (after the last fused step of every rank; the systems themselves stay usable)"""
        if getattr(self, "_links", None) is None:
            return
        self.synchronize()
        for base in getattr(self, "_opened", []):
            self.P.spin_ipc_close(base, 0)
        self._opened, self._links, self._peer = [], None, None

    def iterate_fused(self, n_steps: int) -> None:
        """n fused steps of this rank (every rank calls it with the same n): no halo copy, no message, no host synchronisation"""
        sides = [side for side in (0, 1) if self._peer[side] is not None]
        flags = self._order == "flags"
        # every rank advances in lockstep (copy-based steps in between included), so the neighbours' arrays have the roles this rank's have
        swapped = self.sys.spin_slab_arrays()[0] != self._cur0
        for _ in range(int(n_steps)):
            for op in fused_step_ops(self._fused_step + 1, sides):
                if op[0] == "wait":
                    if flags:
                        self.sys.spin_flag_wait(self._flags + 8 * op[1], op[2])
                elif op[0] == "signal":
                    if flags:
                        self.sys.spin_flag_signal(self._peer[op[1]][2], op[2])
                else:
                    lo, hi = self._peer
                    nxt = 0 if swapped else 1             # the neighbours' NEXT array
                    self.sys.llg_slab_step_fused(lo[nxt] if lo else None, self._links[0].count if lo else 0, hi[nxt] if hi else None)
                    self.sys.llg_slab_advance()
                    swapped = not swapped
            self._fused_step += 1
            if not flags:
                self.synchronize()
                self._dist.barrier(group=self._group)

    def spins(self):
        self.synchronize()
        return self.sys.spins_get()

    def synchronize(self):
        self.copy_stream.synchronize()
        self.sys.spin_synchronize()


class LocalGroup:
    """All slabs of a lattice in ONE process on one device: the emulation of N ranks on one GPU (never run ranks that wait on one another as
    separate launches, B200_PROFILING.md).  The slabs advance in lockstep; a halo message is a device copy from the sender's send buffer
    into the receiver's receive buffer, ordered by the sender's event."""

    def __init__(self, P, torch, w, world: int, options=(), fused: bool = False):
        """fused: steps by llg_slab_step_fused -- every slab's kernel writes its boundary planes straight into its neighbours' ghost layers
        (here: other arrays of the same device; across GPUs: peer memory), no halo copies; needs the one-pass kernel and two slabs or more."""
        self.torch = torch
        self.drivers = [SlabDriver(P, torch, w, r, world, options=options) for r in range(world)]
        self._exchange(0, post=True)
        self.fused = bool(fused) and world >= 2 and all(d.one_pass for d in self.drivers)
        if fused and not self.fused:
            raise ValueError("fused halo exchange needs the one-pass kernel on every slab and at least two slabs")

    def _move(self) -> None:
        for d in self.drivers:
            for side in (0, 1):
                peer = d.plan.neighbour(side)
                if peer is None:
                    continue
                src = self.drivers[peer]
                d.copy_stream.wait_event(src.sent)
                with self.torch.cuda.stream(d.copy_stream):
                    d.recv[side].copy_(src.send[1 - side], non_blocking=True)      # the peer's message towards the opposite side
        # nobody refills a send buffer before every copy out of it has run
        moved = []
        for d in self.drivers:
            ev = self.torch.cuda.Event()
            ev.record(d.copy_stream)
            moved.append(ev)
        for d in self.drivers:
            for ev in moved:
                d.copy_stream.wait_event(ev)

    def _exchange(self, array: int, post: bool) -> None:
        if post:
            for d in self.drivers:
                d.post(array)
        self._move()
        for d in self.drivers:
            d.deliver(array)

    def _iterate_fused(self, n_steps: int) -> None:
        ds, Event = self.drivers, self.torch.cuda.Event
        nxt = [d.sys.spin_slab_arrays() for d in ds]          # (current, next) device addresses; they swap at every advance
        done = []
        for d in ds:                                           # everything enqueued so far (priming copies, earlier steps) is a dependency
            ev = Event(); ev.record(d.stream); done.append(ev)
        for _ in range(int(n_steps)):
            # a slab's step k + 1 needs its neighbours' step k: they wrote its ghost layers, and they read the arrays it now writes into
            for i, d in enumerate(ds):
                for side in (0, 1):
                    p = d.plan.neighbour(side)
                    if p is not None and p != i:
                        d.stream.wait_event(done[p])
            for i, d in enumerate(ds):
                lo, hi = d.plan.neighbour(0), d.plan.neighbour(1)
                d.sys.llg_slab_step_fused(nxt[lo][1] if lo is not None else None, ds[lo].plan.count if lo is not None else 0,
                                          nxt[hi][1] if hi is not None else None)
            for i, d in enumerate(ds):
                d.sys.llg_slab_advance()
                ev = Event(); ev.record(d.stream); done[i] = ev
                nxt[i] = (nxt[i][1], nxt[i][0])

    def iterate(self, n_steps: int) -> None:
        if self.fused:
            return self._iterate_fused(n_steps)
        for _ in range(int(n_steps)):
            plans = [d.stages() for d in self.drivers]      # (every slab is in the same mode: the same Hamiltonian and options)
            for k in range(len(plans[0])):
                for p in plans:
                    p[k][0]()
                self._exchange(plans[0][k][1], post=False)
            for d in self.drivers:
                d.sys.llg_slab_advance()

    def spins(self):
        import numpy as np
        return np.concatenate([d.spins() for d in self.drivers], axis=0)
