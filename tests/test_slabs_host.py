"""Host logic of the slab decomposition (paper_2003_06342_b200/slabs.py) on CPU: ownership, ghost copies, and the two
exchange drivers -- in-process and torch.distributed (gloo, world sizes 2 and 3) -- on a stand-in slab whose "layers"
are tagged with their global index, so that a wrong neighbour, side or message order is visible."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2003_06342_b200 import slabs
from paper_2003_06342_b200 import workloads as wl


def test_split_and_neighbours():
    assert slabs.split_extent(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert slabs.split_extent(8, 1) == [(0, 8)]
    with pytest.raises(ValueError):
        slabs.split_extent(2, 3)
    assert slabs.neighbours(0, 3, False) == (None, 1)
    assert slabs.neighbours(2, 3, False) == (1, None)
    assert slabs.neighbours(0, 3, True) == (2, 1)
    assert slabs.neighbours(0, 1, True) == (0, 0)
    assert slabs.neighbours(0, 1, False) == (None, None)


def test_local_params_walls_3d():
    P, _ = wl.config4_film3d(16, 12, 10)
    P0, P1, P2 = (slabs.local_params(P, r, 3) for r in range(3))
    assert (P0["nz"], P1["nz"], P2["nz"]) == (4 + 1, 3 + 2, 3 + 1)
    assert (P0["halo"], P1["halo"], P2["halo"]) == ((0, 1), (1, 1), (1, 0))
    assert P0["bc_f"][2] == ["wall", "periodic"] and P2["bc_f"][2] == ["periodic", "wall"]
    assert P1["bc_s"][2] == ["periodic", "periodic"] and P0["bc_s"][2][0] == "dirichlet"
    assert P["bc_f"][2] == ["wall", "wall"]                      # the global description is not touched
    assert slabs.local_params(P, 0, 1)["halo"] == (0, 0)


def test_local_params_periodic_2d():
    P, _ = wl.config1_droplet(16)
    assert slabs.slab_axis(P) == 1
    Pl = slabs.local_params(P, 0, 1)
    assert Pl["halo"] == (1, 1) and Pl["ny"] == 18             # a single periodic slab is its own neighbour
    Pl = slabs.local_params(P, 1, 2)
    assert Pl["halo"] == (1, 1) and Pl["ny"] == 10 and Pl["slab"]["start"] == 8


def test_local_block_and_strip():
    P, _ = wl.config5_droplets(6, nspheres=1, rmin=1.0, rmax=2.0)
    a = np.arange(6 * 6 * 6, dtype=float).reshape(6, 6, 6)
    b = slabs.local_block(a, P, 0, 2)                              # layers -1..3 -> 5, 0, 1, 2, 3
    assert b.shape == (5, 6, 6)
    assert np.array_equal(b[:, 0, 0], a[[5, 0, 1, 2, 3], 0, 0])
    u = np.stack([a, 2 * a, 3 * a])
    bu = slabs.local_block(u, P, 1, 2)                             # layers 2..6 -> 2, 3, 4, 5, 0
    assert np.array_equal(bu[1, :, 0, 0], 2 * a[[2, 3, 4, 5, 0], 0, 0])
    Pl = slabs.local_params(P, 1, 2)
    assert np.array_equal(slabs.strip_ghosts(bu, Pl), u[:, 3:6])
    P2, _ = wl.config3_film2d(8, 9)                                # 2D: cut along y, walls at the ends
    a2 = np.arange(9 * 8, dtype=float).reshape(1, 9, 8)
    assert np.array_equal(slabs.local_block(a2, P2, 1, 2)[0, :, 0], a2[0, 4:9, 0])   # rows 4..8: ghost 4, owned 5..8


def test_layer_parts():
    assert slabs.layer_parts(10, (1, 1)) == {"boundary": [(1, 1), (8, 1)], "interior": (2, 6)}
    assert slabs.layer_parts(10, (0, 1)) == {"boundary": [(8, 1)], "interior": (0, 8)}          # physical face below
    assert slabs.layer_parts(10, (1, 0)) == {"boundary": [(1, 1)], "interior": (2, 8)}
    assert slabs.layer_parts(3, (1, 1)) == {"boundary": [(1, 1)], "interior": (2, 0)}           # one owned layer
    assert slabs.layer_parts(4, (1, 1)) == {"boundary": [(1, 1), (2, 1)], "interior": (2, 0)}   # two owned layers
    assert slabs.layer_parts(6, (0, 0)) == {"boundary": [], "interior": (0, 6)}
    for n, halo in ((10, (1, 1)), (10, (0, 1)), (3, (1, 1)), (4, (1, 1)), (5, (1, 0)), (2, (0, 1))):   # every owned layer once
        parts = slabs.layer_parts(n, halo)
        got = sorted(l for f, c in parts["boundary"] + [parts["interior"]] for l in range(f, f + c))
        assert got == list(range(halo[0], n - halo[1])), (n, halo, parts)


class TaggedSlab:
    """Stand-in for slabs.Slab: one number per layer.  ``layers`` holds the global layer index of every local layer
    (ghosts start at -1); pack/unpack move [layer id, what, sender side] so that the test can see who sent what."""

    def __init__(self, n_global, rank, world, periodic):
        start, count = slabs.split_extent(n_global, world)[rank]
        lo, hi = slabs.neighbours(rank, world, periodic)
        self.halo = (0 if lo is None else 1, 0 if hi is None else 1)
        self.layers = [-1] * self.halo[0] + list(range(start, start + count)) + [-1] * self.halo[1]
        self.seen = {}
        self.log = []
        self._send = {w: {s: torch.zeros(3, dtype=torch.int64) for s in range(2) if self.halo[s]} for w in range(2)}
        self._recv = {w: {s: torch.zeros(3, dtype=torch.int64) for s in range(2) if self.halo[s]} for w in range(2)}

    def buffers(self, what):
        return self._send[what]

    def recv_buffers(self, what):
        return self._recv[what]

    def halo_pack(self, what, side, buf):
        owned = self.layers[1] if side == 0 else self.layers[-2]
        buf.copy_(torch.tensor([owned, what, side]))
        self.log.append(("pack", what, side))

    def halo_unpack(self, what, side, buf):
        layer, w, sender_side = (int(v) for v in buf)
        assert w == what and sender_side == 1 - side
        self.layers[0 if side == 0 else -1] = layer
        self.seen[(what, side)] = layer
        self.log.append(("unpack", what, side))

    # overlapped schedule (slabs.step_overlapped): what ran, in host order
    log = None

    def run_part(self, phase, which, store_macros, last):
        self.log.append(("part", phase, which, bool(store_macros), bool(last)))


def _expected_layers(n_global, rank, world, periodic):
    start, count = slabs.split_extent(n_global, world)[rank]
    lo, hi = slabs.neighbours(rank, world, periodic)
    out = list(range(start, start + count))
    if lo is not None:
        out = [(start - 1) % n_global] + out
    if hi is not None:
        out = out + [(start + count) % n_global]
    return out


@pytest.mark.parametrize("world,periodic", [(1, True), (2, True), (3, True), (2, False), (4, False)])
def test_exchange_local(world, periodic):
    n = 11
    S = [TaggedSlab(n, r, world, periodic) for r in range(world)]
    for what in (slabs.HALO_POPS, slabs.HALO_PHI):
        slabs.exchange_local(S, what, periodic)
    for r, s in enumerate(S):
        assert s.layers == _expected_layers(n, r, world, periodic)


def _expected_log(halo, nsteps):
    """Host order of the overlapped schedule for one slab: boundary part, exchange, interior part -- per phase."""
    sides = [s for s in range(2) if halo[s]]
    out = []
    for k in range(nsteps):
        macro = k == nsteps - 1
        for phase, what in ((0, slabs.HALO_PHI), (1, slabs.HALO_POPS)):
            m = macro and phase == 1
            out.append(("part", phase, "boundary", m, False))
            out += [("pack", what, s) for s in sides] + [("unpack", what, s) for s in sides]
            out.append(("part", phase, "interior", m, True))
    return out


@pytest.mark.parametrize("world,periodic", [(1, True), (3, True), (3, False)])
def test_step_overlapped_local_order(world, periodic):
    n = 11
    S = [TaggedSlab(n, r, world, periodic) for r in range(world)]
    slabs.step_overlapped(S, lambda what: slabs.exchange_local(S, what, periodic), slabs.NoStreams(), 2)
    for r, s in enumerate(S):
        assert s.layers == _expected_layers(n, r, world, periodic)
        assert s.log == _expected_log(s.halo, 2), (r, s.log)


def _worker_overlapped(rank, world, port, periodic, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s = TaggedSlab(11, rank, world, periodic)
    slabs.step_overlapped([s], lambda what: slabs.exchange_dist(s, what, rank, world, periodic), slabs.NoStreams(), 3)
    out.put((rank, (s.layers, s.log == _expected_log(s.halo, 3))))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True)])
def test_step_overlapped_dist_gloo(world, periodic):
    """The boundary-first schedule over torch.distributed (gloo): two exchanges per step between the parts of a phase, three
    steps in a row -- messages of consecutive exchanges to the same peer must not cross-match (world 2, periodic: both
    neighbours are the same rank)."""
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker_overlapped, args=(r, world, port, periodic, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert res[r][0] == _expected_layers(11, r, world, periodic), (r, res[r])
        assert res[r][1], "rank %d: parts and exchanges out of order" % r


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, periodic, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s = TaggedSlab(11, rank, world, periodic)
    for _ in range(3):                                   # repeated exchanges must not cross-match messages
        for what in (slabs.HALO_PHI, slabs.HALO_POPS):
            slabs.exchange_dist(s, what, rank, world, periodic)
    out.put((rank, s.layers))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True)])
def test_exchange_dist_gloo(world, periodic):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, periodic, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        assert res[r] == _expected_layers(11, r, world, periodic), (r, res[r])
