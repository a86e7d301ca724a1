"""Slab decomposition of one domain over several contexts (the paper's multi-GPU mode).

The domain is cut along its SLOWEST axis (z in 3D, y in 2D) into contiguous slabs.  Each slab is an ordinary context of
the C ABI whose parameters declare a ghost layer on every cut side (``lbm_params.halo``, include/lbm.h); a step is

    K_phi (phase 0)  ->  exchange LBM_HALO_PHI  ->  K_main (phase 1)  ->  exchange LBM_HALO_POPS

and the exchanges move one padded phi layer and the 7 (3D) populations that cross the cut, per side.  Everything the
method computes still runs in the kernels; this module only decides who owns which layers and moves the packed buffers:

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

    def __init__(self, P: dict, nslabs: int, precision: int = 64):
        import torch
        self.P = P
        self.periodic = axis_is_periodic(P)
        self.stream = torch.cuda.Stream()   # one stream for all slabs: pack, hand-over and unpack are ordered by it
        self.slabs = [Slab(P, r, nslabs, precision, stream=self.stream) for r in range(nslabs)]
        self.any_halo = any(s.has_halo for s in self.slabs)

    def init(self, phi, T=None, u=None, p=None):
        for s in self.slabs:
            s.init(phi, T, u, p)
        if self.any_halo:
            exchange_local(self.slabs, HALO_POPS, self.periodic)   # ghost populations of level 0

    def step(self, n: int = 1):
        if not self.any_halo:
            self.slabs[0].sim.step(n)
            return
        for k in range(n):
            for s in self.slabs:
                s.sim.step_phase(0)
            exchange_local(self.slabs, HALO_PHI, self.periodic)
            for s in self.slabs:
                s.sim.step_phase(1, store_macros=(k == n - 1))
            exchange_local(self.slabs, HALO_POPS, self.periodic)

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

    def __init__(self, P: dict, rank: int, world: int, precision: int = 64, group=None):
        self.periodic = axis_is_periodic(P)
        import torch
        self.rank, self.world, self.group = rank, world, group
        # the transfers (torch.distributed) are enqueued on torch's current stream: the slab's kernels go there too
        self.slab = Slab(P, rank, world, precision, stream=torch.cuda.current_stream())

    def init(self, phi, T=None, u=None, p=None, local=False):
        """GLOBAL fields, or with ``local=True`` this rank's layers including the ghost copies (Slab.layer_range)."""
        (self.slab.init_local if local else self.slab.init)(phi, T, u, p)
        if self.slab.has_halo:
            exchange_dist(self.slab, HALO_POPS, self.rank, self.world, self.periodic, self.group)

    def step(self, n: int = 1):
        s = self.slab
        if not s.has_halo:
            s.sim.step(n)
            return
        for k in range(n):
            s.sim.step_phase(0)
            exchange_dist(s, HALO_PHI, self.rank, self.world, self.periodic, self.group)
            s.sim.step_phase(1, store_macros=(k == n - 1))
            exchange_dist(s, HALO_POPS, self.rank, self.world, self.periodic, self.group)

    def read_macro(self):
        """Owned layers of this rank (no gather: results stay sharded)."""
        return self.slab.read_macro()

    def destroy(self):
        self.slab.destroy()
