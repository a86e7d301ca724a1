"""Slab decomposition of one domain over several contexts (the paper's multi-GPU mode).

The domain is cut along its SLOWEST axis (z in 3D, y in 2D) into contiguous slabs.  Each slab is an ordinary context of
the C ABI whose parameters declare a ghost layer on every cut side (``lbm_params.halo``, include/lbm.h); a step is

    K_phi (phase 0)  ->  exchange LBM_HALO_PHI  ->  K_main (phase 1)  ->  exchange LBM_HALO_POPS

and the exchanges move one padded phi layer and the 7 (3D) populations that cross the cut, per side.  The default schedule
overlaps them with the interior (:func:`step_overlapped`: boundary layers first on the compute stream, pack / transfer /
unpack on a second stream, ordered by events; the ghost layers themselves are never computed); ``overlap=False`` keeps the
plain one-stream sequence above.  Everything the method computes still runs in the kernels; this module only decides who owns
which layers and moves the packed buffers:

* :class:`SlabGroup`  -- all slabs in ONE process on one GPU (the buffers are handed over directly); this is how the
  decomposition is parity-tested on a single GPU (tests/test_gpu_slabs.py): the stitched result equals the undecomposed
  run -- bit for bit on periodic domains, to rounding where physical faces select the boundary instantiation;
* :class:`DistSlab`   -- one slab per rank, buffers moved with ``torch.distributed`` point-to-point calls (NCCL over
  NVLink on GPUs; the same code runs over ``gloo`` with CPU buffers in tests/test_slabs_host.py).

No arithmetic of the method lives here.
"""
from __future__ import annotations

import copy

import numpy as np

HALO_PHI, HALO_POPS = 0, 1
PERIODIC = "periodic"


# ---------------------------------------------------------------------------------------------- ownership (host logic)
def slab_axis(P: dict) -> int:
    """Physical axis the domain is cut along: 2 (z) in 3D, 1 (y) in 2D."""
    return 2 if int(P.get("nz", 1)) > 1 else 1


def _axis_key(P):
    return "nz" if slab_axis(P) == 2 else "ny"


def axis_is_periodic(P: dict) -> bool:
    return P["bc_f"][slab_axis(P)][0] == PERIODIC


def split_extent(n: int, parts: int):
    """[(start, count)] of ``parts`` contiguous slabs covering 0..n-1; the first n % parts slabs get one more layer."""
    if parts < 1 or n < parts:
        raise ValueError("cannot cut %d layers into %d slabs" % (n, parts))
    base, rem = divmod(n, parts)
    out, s = [], 0
    for r in range(parts):
        c = base + (1 if r < rem else 0)
        out.append((s, c))
        s += c
    return out


def neighbours(rank: int, world: int, periodic: bool):
    """(rank below, rank above) along the slab axis; None where the slab ends on a physical face."""
    lo = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    hi = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return lo, hi


def local_params(P: dict, rank: int, world: int) -> dict:
    """Parameters of slab ``rank``: its layers plus one ghost layer per cut side; cut faces become periodic-kind."""
    ax, key = slab_axis(P), _axis_key(P)
    start, count = split_extent(int(P[key]), world)[rank]
    lo, hi = neighbours(rank, world, axis_is_periodic(P))
    halo = (0 if lo is None else 1, 0 if hi is None else 1)
    Pl = copy.deepcopy(P)
    Pl[key] = count + halo[0] + halo[1]
    Pl["halo"] = halo
    Pl["slab"] = dict(rank=rank, world=world, start=start, count=count, axis=ax)
    for side in range(2):
        if halo[side]:
            for k in ("bc_f", "bc_g", "bc_s"):
                Pl[k][ax][side] = PERIODIC
    return Pl


def _array_axis(P, a):
    """numpy axis of the slab axis in an array shaped (nz, ny, nx) or (C, nz, ny, nx)."""
    return (0 if slab_axis(P) == 2 else 1) + (a.ndim - 3)


def local_block(a, P: dict, rank: int, world: int):
    """Layers of the global array ``a`` that slab ``rank`` holds, ghost layers included (periodic wrap across the ends)."""
    if a is None:
        return None
    a = np.asarray(a)
    Pl = local_params(P, rank, world)
    s = Pl["slab"]
    idx = np.arange(s["start"] - Pl["halo"][0], s["start"] + s["count"] + Pl["halo"][1])
    return np.ascontiguousarray(np.take(a, idx, axis=_array_axis(P, a), mode="wrap"))


def strip_ghosts(a, Pl: dict):
    """Owned layers of a slab-local array."""
    ax = _array_axis(Pl, a)
    n = a.shape[ax]
    sl = [slice(None)] * a.ndim
    sl[ax] = slice(Pl["halo"][0], n - Pl["halo"][1])
    return a[tuple(sl)]


# ---------------------------------------------------------------------------------------------------------- exchange
def exchange_local(slabs, what: int, periodic: bool):
    """All slabs in one process: every slab packs its cut sides, then every slab unpacks its neighbours' buffers.

    ``slabs[r]`` offers ``halo``, ``buffers(what)`` -> {side: tensor}, ``halo_pack`` and ``halo_unpack``."""
    world = len(slabs)
    for sl in slabs:
        for side in range(2):
            if sl.halo[side]:
                sl.halo_pack(what, side, sl.buffers(what)[side])
    for r, sl in enumerate(slabs):
        nb = neighbours(r, world, periodic)
        for side in range(2):
            if sl.halo[side]:
                # my ghost layer of `side` mirrors the neighbour's boundary layer of the opposite side
                sl.halo_unpack(what, side, slabs[nb[side]].buffers(what)[1 - side])


def exchange_push(slabs, what: int, periodic: bool):
    """All slabs in one process on one GPU (or with peer-mapped workspaces): every cut side is ONE launch that copies the
    boundary layer straight into the neighbour's ghost layer (lbm_halo_push) -- no buffers, no unpack."""
    world = len(slabs)
    for r, sl in enumerate(slabs):
        nb = neighbours(r, world, periodic)
        for side in range(2):
            if sl.halo[side]:
                sl.halo_push(what, side, slabs[nb[side]])


def exchange_push_mapped(slabs, what: int, periodic: bool):
    """As :func:`exchange_push`, with the neighbour known only by its parameters and the device address of its workspace
    (lbm_halo_push_mapped) -- the form a multi-process run takes once the workspaces are peer-mapped (CUDA IPC); here the
    "mapped" address is simply the neighbour's own, which is how the call is tested on one GPU."""
    world = len(slabs)
    for r, sl in enumerate(slabs):
        nb = neighbours(r, world, periodic)
        for side in range(2):
            if sl.halo[side]:
                peer = slabs[nb[side]]
                sl.sim.halo_push_mapped(what, side, peer.P, peer.sim.workspace_ptr)


def exchange_dist(slab, what: int, rank: int, world: int, periodic: bool, group=None):
    """One slab per rank: pack, post all sends and receives as one batch, wait, unpack.

    The message packed on the sender's ``side`` lands in the receiver's ``1 - side`` ghost layer.  Tags carry the
    sender's side; the receives are posted in the order of the peer's sends so that backends which match messages of
    one pair of ranks by order only (NCCL) pair them correctly when both neighbours are the same rank (world = 2)."""
    import torch.distributed as dist
    nb = neighbours(rank, world, periodic)
    send = slab.buffers(what)
    recv = slab.recv_buffers(what)
    for side in range(2):
        if slab.halo[side]:
            slab.halo_pack(what, side, send[side])
    ops = []
    for side in range(2):
        if slab.halo[side] and nb[side] != rank:
            ops.append(dist.P2POp(dist.isend, send[side], nb[side], group=group, tag=side))
    for side in (1, 0):   # the peer sends side 0 first, which arrives in MY side 1
        if slab.halo[side] and nb[side] != rank:
            ops.append(dist.P2POp(dist.irecv, recv[side], nb[side], group=group, tag=1 - side))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    for side in range(2):
        if slab.halo[side]:
            src = recv[side] if nb[side] != rank else send[1 - side]   # a single periodic slab is its own neighbour
            slab.halo_unpack(what, side, src)


class PeerTransport:
    """Ghost-layer exchange of one slab per process WITHOUT a communication library: every process maps its neighbours'
    workspaces through CUDA IPC (the handles travel once, over ``torch.distributed`` object collectives) and pushes its boundary
    layers straight into their ghost layers (lbm_halo_push_mapped: one copy kernel per cut side and phase, stores over
    NVLink / peer memory).  Ordering, ``sync="flags"`` (the default): after its pushes a rank enqueues the write of the exchange's
    sequence number into a word of the neighbour's (mapped) memory, and enqueues a wait on its own word for the neighbour's --
    stream memory operations of the driver (lbm_stream_signal / lbm_stream_wait): nothing on the host waits and no kernel spins.
    ``sync="events"``: an inter-process event per exchange kind and a host barrier that makes sure every rank has recorded before
    anybody enqueues the wait (a wait captures the latest record at the time of the call).  In both, the double-buffered
    populations and phi arrays keep a push of step n + 1 off the layers step n still reads."""

    def __init__(self, slab, rank: int, world: int, periodic: bool, group=None, sync: str = "flags"):
        import torch
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        self.slab, self.rank, self.world, self.sync = slab, rank, world, sync
        # the handles and the barriers are host business: a gloo group beside an NCCL job (an NCCL barrier would stall the stream)
        self.group = group if dist.get_backend(group) == "gloo" else dist.new_group(backend="gloo")
        group = self.group
        self.nb = neighbours(rank, world, periodic)
        dev = torch.cuda.current_device()
        self.flags = torch.zeros(4, dtype=torch.int32, device="cuda")     # word [2 * what + side]: last exchange received there
        self.seq = {HALO_PHI: 0, HALO_POPS: 0}
        self.done = {what: torch.cuda.Event(enable_timing=False, interprocess=True) for what in (HALO_PHI, HALO_POPS)}
        for ev in self.done.values():
            ev.record(slab.sim.stream)                  # the CUDA event exists from its first record on
        torch.cuda.synchronize()
        mine = {"ws": reduce_tensor(slab.sim.workspace_tensor), "flags": reduce_tensor(self.flags), "P": slab.P,
                "ev": {what: ev.ipc_handle() for what, ev in self.done.items()}}
        infos = [None] * world
        dist.all_gather_object(infos, mine, group=group)
        self.peer_ws, self.peer_flags, self.peer_P, self.peer_ev = {}, {}, {}, {}
        for side in range(2):
            if slab.halo[side] and self.nb[side] != rank:
                info = infos[self.nb[side]]
                rebuild, args = info["ws"]
                self.peer_ws[side] = rebuild(*args)      # the neighbour's workspace, mapped into this process
                rebuild, args = info["flags"]
                self.peer_flags[side] = rebuild(*args)
                self.peer_P[side] = info["P"]
                self.peer_ev[side] = {what: torch.cuda.Event.from_ipc_handle(dev, h) for what, h in info["ev"].items()}

    def ready(self):
        """Host barrier (once, after lbm_init, which writes the ghost layers too): nobody pushes into a workspace still being set up."""
        import torch.distributed as dist
        dist.barrier(group=self.group)

    def exchange(self, what: int):
        """On torch's CURRENT stream (the slab's calls are enqueued there too): push, signal, wait."""
        import torch
        import torch.distributed as dist
        s = self.slab
        st = torch.cuda.current_stream()
        self.seq[what] += 1
        seq = self.seq[what]
        for side in range(2):
            if not s.halo[side]:
                continue
            if self.nb[side] == self.rank:
                s.sim.halo_push(what, side, s.sim)       # a single periodic slab is its own neighbour
            else:
                s.sim.halo_push_mapped(what, side, self.peer_P[side], self.peer_ws[side].data_ptr())
                if self.sync == "flags":                 # my push lands in the neighbour's ghost layer of the OPPOSITE side
                    s.sim.stream_signal(self.peer_flags[side].data_ptr() + 4 * (2 * what + (1 - side)), seq)
        if self.sync == "flags":
            for side in range(2):
                if s.halo[side] and self.nb[side] != self.rank:
                    s.sim.stream_wait(self.flags.data_ptr() + 4 * (2 * what + side), seq)
            return
        self.done[what].record(st)
        dist.barrier(group=self.group)                   # host: everybody has enqueued its pushes and recorded
        for side in range(2):
            if s.halo[side] and self.nb[side] != self.rank:
                st.wait_event(self.peer_ev[side][what])  # my ghost layer of `side` was written by that neighbour


# ------------------------------------------------------------------------------------------- overlapped schedule (host logic)
def layer_parts(n_local: int, halo):
    """Owned layers of a slab with ``n_local`` layers (ghosts included) by role: ``boundary`` = [(first, count)] of the owned
    layers next to a ghost layer (what the neighbours wait for), ``interior`` = (first, count) of the other owned layers."""
    lo, hi = halo[0], n_local - halo[1]                 # owned layers [lo, hi)
    boundary = []
    if halo[0]:
        boundary.append((lo, 1))
    if halo[1] and (hi - 1 != lo or not halo[0]):
        boundary.append((hi - 1, 1))
    first = lo + (1 if halo[0] else 0)
    last = hi - (1 if halo[1] else 0)
    return {"boundary": boundary, "interior": (first, max(last - first, 0))}


class NoStreams:
    """Stand-in for :class:`TwoStreams` where everything is ordered by the host (CPU tests)."""

    def begin_exchange(self, slabs):
        pass

    def end_exchange(self, slabs):
        pass

    def wait_exchange(self):
        pass

    def exchange_context(self):
        import contextlib
        return contextlib.nullcontext()


class TwoStreams:
    """Compute stream C and exchange stream X (pack, transfer, unpack, and K_main of the boundary layers), ordered by events:
    X continues after what C has enqueued so far (begin_exchange); C waits for X where it needs its results (wait_exchange)."""

    def __init__(self, compute, exchange):
        self.C, self.X, self.pending = compute, exchange, None

    def begin_exchange(self, slabs):
        import torch
        ev = torch.cuda.Event()
        ev.record(self.C)
        self.X.wait_event(ev)
        for s in slabs:
            s.set_stream(self.X)

    def end_exchange(self, slabs):
        import torch
        self.pending = torch.cuda.Event()
        self.pending.record(self.X)
        for s in slabs:
            s.set_stream(self.C)

    def wait_exchange(self):
        if self.pending is not None:
            self.C.wait_event(self.pending)
            self.pending = None

    def exchange_context(self):
        import torch
        return torch.cuda.stream(self.X)        # torch.distributed orders its transfers against the CURRENT stream


def step_overlapped(slabs, exchange, sched, n: int, macros: bool = True):
    """``n`` steps of the slabs of this process, boundary layers first, on two streams:

        C:  K_phi(boundary) . K_phi(interior) ............ K_main(interior) ............................ | next step
        X:                  . exchange phi    . K_main(boundary) . exchange populations ............... -^

    C is the compute stream, X the exchange stream (higher priority).  K_main of the boundary layers -- less than one wave of
    CTAs -- runs on X while the interior fills the SMs on C; the next step on C waits for X once, at its start.
    ``slabs[i].run_part(phase, which, store_macros, last)`` enqueues one part on the slab's current stream, ``exchange(what)``
    packs, moves and unpacks, ``sched`` switches the slabs between the streams and orders these with events."""
    for k in range(n):
        macro = macros and k == n - 1                      # u, p, T are stored by the last step of a call (not inside a graph)
        sched.wait_exchange()                              # boundary layers and ghost populations of the previous level
        for s in slabs:
            s.run_part(0, "boundary", False, False)
        sched.begin_exchange(slabs)                        # X: after K_phi(boundary)
        with sched.exchange_context():
            exchange(HALO_PHI)
        sched.end_exchange(slabs)
        for s in slabs:
            s.run_part(0, "interior", False, True)
        sched.begin_exchange(slabs)                        # X: after K_phi(interior) as well
        for s in slabs:
            s.run_part(1, "boundary", macro, False)
        with sched.exchange_context():
            exchange(HALO_POPS)
        sched.end_exchange(slabs)
        for s in slabs:
            s.run_part(1, "interior", macro, True)
    sched.wait_exchange()


# ------------------------------------------------------------------------------------------------------ slab contexts
class Slab:
    """One slab context plus its exchange buffers.  Device memory comes from torch (plumbing)."""

    def __init__(self, P: dict, rank: int, world: int, precision: int = 64, stream=None):
        import torch
        from . import binding
        self.Pg = P
        self.P = local_params(P, rank, world)
        self.rank, self.world = rank, world
        self.halo = self.P["halo"]
        self.has_halo = bool(self.halo[0] or self.halo[1])
        self.sim = binding.LBM(self.P, precision, stream=stream)
        self._send, self._recv = {}, {}
        if self.has_halo:
            for what in (HALO_PHI, HALO_POPS):
                n = self.sim.halo_bytes(what)
                self._send[what] = {s: torch.empty(n, dtype=torch.uint8, device="cuda") for s in range(2) if self.halo[s]}
                self._recv[what] = {s: torch.empty(n, dtype=torch.uint8, device="cuda") for s in range(2) if self.halo[s]}

    def buffers(self, what):
        return self._send[what]

    def recv_buffers(self, what):
        return self._recv[what]

    def halo_pack(self, what, side, buf):
        self.sim.halo_pack(what, side, buf)

    def halo_unpack(self, what, side, buf):
        self.sim.halo_unpack(what, side, buf)

    def halo_push(self, what, side, peer):
        self.sim.halo_push(what, side, peer.sim)

    def set_stream(self, stream):
        self.sim.set_stream(stream)

    def run_part(self, phase, which, store_macros, last):
        """One part of a phase (lbm_step_layers): the owned layers next to the ghost layers, or the other owned layers."""
        n = int(self.P["nz"]) if slab_axis(self.P) == 2 else int(self.P["ny"])
        parts = layer_parts(n, self.halo)
        ranges = parts["boundary"] if which == "boundary" else [parts["interior"]]
        if not ranges:
            ranges = [(0, 0)]
        for i, (first, count) in enumerate(ranges):
            self.sim.step_layers(phase, first, count, store_macros, last and i == len(ranges) - 1)

    def init(self, phi, T=None, u=None, p=None):
        """GLOBAL initial fields; the slab takes its layers and the ghost copies."""
        args = [local_block(a, self.Pg, self.rank, self.world) for a in (phi, T, u, p)]
        self.sim.init(*args)

    def init_local(self, phi, T=None, u=None, p=None):
        """The slab's own layers INCLUDING the ghost copies (``layer_range``), for domains too large to build whole."""
        self.sim.init(phi, T, u, p)

    def layer_range(self):
        """(first, last + 1) global layer index of the local arrays, ghost layers included (no wrap: may leave 0..n-1
        on a periodic axis)."""
        s = self.P["slab"]
        return s["start"] - self.halo[0], s["start"] + s["count"] + self.halo[1]

    def read_macro(self):
        return tuple(strip_ghosts(a, self.P) for a in self.sim.read_macro())

    def read_pops(self, which, stage):
        return strip_ghosts(self.sim.read_pops(which, stage), self.P)

    def destroy(self):
        self.sim.destroy()


class SlabGroup:
    """``nslabs`` slabs of one domain in one process, on the current device and stream."""

    def __init__(self, P: dict, nslabs: int, precision: int = 64, overlap: bool = True, graph: bool = True, push: bool = True):
        import torch
        self.P = P
        # the slabs share a GPU: a boundary layer goes straight into the neighbour's ghost layer (one launch per cut side and
        # phase) instead of pack -> buffer -> unpack (two); push=False keeps the buffered exchange a multi-process run uses
        self._exchange = exchange_push_mapped if push == "mapped" else (exchange_push if push else exchange_local)
        # the overlapped step of small slabs is launch-bound (fourteen short launches per slab and step): replay it from a CUDA
        # graph of two consecutive steps (the buffers alternate with period 2), captured across both streams, one per parity
        self.graph = graph
        self._graphs = {}
        self.periodic = axis_is_periodic(P)
        self.stream = torch.cuda.Stream()   # compute stream of all slabs
        self.slabs = [Slab(P, r, nslabs, precision, stream=self.stream) for r in range(nslabs)]
        self.any_halo = any(s.has_halo for s in self.slabs)
        self.overlap = overlap and not P.get("prescribed_u", False)
        self.sched = TwoStreams(self.stream, torch.cuda.Stream(priority=-1)) if self.overlap else None

    def init(self, phi, T=None, u=None, p=None):
        for s in self.slabs:
            s.init(phi, T, u, p)
        if self.any_halo:
            self._exchange(self.slabs, HALO_POPS, self.periodic)   # ghost populations of level 0

    def step(self, n: int = 1):
        if not self.any_halo:
            self.slabs[0].sim.step(n)
            return
        if self.overlap:
            exch = lambda what: self._exchange(self.slabs, what, self.periodic)   # noqa: E731
            plain = n - 1
            small = max(s.sim.N for s in self.slabs) <= (1 << 21)
            if self.graph and small and plain >= 6:
                if self.slabs[0].sim.step_count < 2:      # every kernel has been launched once (attributes set) before a capture
                    step_overlapped(self.slabs, exch, self.sched, 2, macros=False)
                    plain -= 2
                plain -= self._replay(plain // 2, exch)
            if plain > 0:
                step_overlapped(self.slabs, exch, self.sched, plain, macros=False)
            step_overlapped(self.slabs, exch, self.sched, 1)
            return
        for k in range(n):
            for s in self.slabs:
                s.sim.step_phase(0)
            self._exchange(self.slabs, HALO_PHI, self.periodic)
            for s in self.slabs:
                s.sim.step_phase(1, store_macros=(k == n - 1))
            self._exchange(self.slabs, HALO_POPS, self.periodic)

    def _replay(self, pairs: int, exch) -> int:
        """``pairs`` times two plain steps from the CUDA graph of the current buffer parity; returns the steps done."""
        import torch
        parity = self.slabs[0].sim.step_count & 1
        if parity not in self._graphs:
            torch.cuda.synchronize()
            before = [(s.sim.step_count, s.sim.launch_count) for s in self.slabs]
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=self.stream):
                step_overlapped(self.slabs, exch, self.sched, 2, macros=False)
            # capture only records: nothing ran, the contexts' counters go back; a replay then advances them
            per = [(s.sim.step_count - b[0], s.sim.launch_count - b[1]) for s, b in zip(self.slabs, before)]
            for s, d in zip(self.slabs, per):
                s.sim.note_replay(-d[0], -d[1])
            self._graphs[parity] = (g, per)
        g, per = self._graphs[parity]
        with torch.cuda.stream(self.stream):
            for _ in range(pairs):
                g.replay()
        for s, d in zip(self.slabs, per):
            s.sim.note_replay(d[0] * pairs, d[1] * pairs)
        return 2 * pairs

    def _stitch(self, parts):
        return np.concatenate(parts, axis=_array_axis(self.P, parts[0]))

    def read_macro(self):
        per = [s.read_macro() for s in self.slabs]
        return tuple(self._stitch([p[i] for p in per]) for i in range(4))

    def read_pops(self, which, stage):
        return self._stitch([s.read_pops(which, stage) for s in self.slabs])

    def destroy(self):
        for s in self.slabs:
            s.destroy()


class DistSlab:
    """The slab of this rank in a ``torch.distributed`` job (one process per GPU)."""

    def __init__(self, P: dict, rank: int, world: int, precision: int = 64, group=None, overlap: bool = True,
                 transport: str = "p2p", peer_sync: str = "flags"):
        """``transport``: "p2p" -- pack, ``torch.distributed`` point-to-point calls (NCCL over NVLink), unpack; "peer" -- the
        neighbours' workspaces mapped through CUDA IPC and written directly (:class:`PeerTransport`; same node only)."""
        self.periodic = axis_is_periodic(P)
        import torch
        self.rank, self.world, self.group = rank, world, group
        self.transport = transport
        self.overlap = overlap and not P.get("prescribed_u", False)
        if self.overlap:
            # kernels on a compute stream of the slab's own; packs, transfers and unpacks on the exchange stream
            self.slab = Slab(P, rank, world, precision)
            self.stream = self.slab.sim.stream
            self.sched = TwoStreams(self.stream, torch.cuda.Stream(priority=-1))
        else:
            # the transfers (torch.distributed) are enqueued on torch's current stream: the slab's kernels go there too
            self.stream = torch.cuda.current_stream()
            self.slab = Slab(P, rank, world, precision, stream=self.stream)
            self.sched = None
        if transport == "peer" and not self.overlap:
            # the plain schedule lets K_main run over the ghost layers and relies on the unpack that follows it in the SAME stream
            # to overwrite the result; a neighbour's push from another process is not ordered against that kernel
            raise ValueError("the peer transport needs the overlapped schedule (ghost layers are never computed there)")
        self.peer = (PeerTransport(self.slab, rank, world, self.periodic, group, sync=peer_sync)
                     if transport == "peer" and self.slab.has_halo else None)

    def _exchange(self, what):
        if self.peer is not None:
            self.peer.exchange(what)
        else:
            exchange_dist(self.slab, what, self.rank, self.world, self.periodic, self.group)

    def init(self, phi, T=None, u=None, p=None, local=False):
        """GLOBAL fields, or with ``local=True`` this rank's layers including the ghost copies (Slab.layer_range)."""
        import torch
        (self.slab.init_local if local else self.slab.init)(phi, T, u, p)
        if self.peer is not None:
            self.peer.ready()                        # lbm_init has finished everywhere (it writes the ghost layers too) before anybody pushes
        if self.slab.has_halo:
            with torch.cuda.stream(self.stream):     # packs, transfers and unpacks of level 0 on the compute stream
                self._exchange(HALO_POPS)

    def step(self, n: int = 1):
        import torch
        s = self.slab
        if not s.has_halo:
            s.sim.step(n)
            return
        if self.overlap:
            step_overlapped([s], self._exchange, self.sched, n)
            return
        with torch.cuda.stream(self.stream):
            for k in range(n):
                s.sim.step_phase(0)
                self._exchange(HALO_PHI)
                s.sim.step_phase(1, store_macros=(k == n - 1))
                self._exchange(HALO_POPS)

    def read_macro(self):
        """Owned layers of this rank (no gather: results stay sharded)."""
        return self.slab.read_macro()

    def destroy(self):
        self.slab.destroy()
