"""DistSlab with the "peer" transport: one slab per PROCESS, the neighbours' workspaces mapped through CUDA IPC and written
directly by lbm_halo_push_mapped; ordering by stream memory operations on flags in mapped memory (lbm_stream_signal / lbm_stream_wait:
no host synchronisation at all) or by inter-process events and a host barrier -- no communication library on the data path.  CUDA IPC
works between two processes on ONE device as well, so this is the multi-process slab path running on the one GPU available:
two processes, both on cuda:0, against the whole-domain oracle.  (What it cannot show is NVLink: on one GPU the "peer" memory is
local.  No kernel waits on another one -- the ordering is stream waits on events -- so the two processes merely time-slice.)"""
import os
import socket

import numpy as np
import pytest

from paper_2003_06342_b200 import workloads as wl
from test_oracle_bruteforce import _random_state

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, P, init, sync, precision, nsteps, out):
    import torch
    import torch.distributed as dist
    from paper_2003_06342_b200 import slabs
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(0)                       # every rank on the same device
    dist.init_process_group("gloo", rank=rank, world_size=world)     # host collectives only: handles, barriers
    dt = np.float64 if precision == 64 else np.float32
    sim = slabs.DistSlab(P, rank, world, precision, overlap=True, transport="peer", peer_sync=sync)
    sim.init(*[None if a is None else a.astype(dt) for a in init])
    sim.step(3)
    sim.step(nsteps - 3)
    out.put((rank, [np.asarray(a) for a in sim.read_macro()]))
    dist.barrier()                                 # nobody unmaps a workspace a neighbour may still write
    sim.destroy()
    dist.destroy_process_group()


@pytest.mark.parametrize("case", ["periodic", "walls", "walls-fp32", "periodic-3ranks", "periodic-events", "walls-events"])
def test_peer_transport_two_processes_one_gpu(oracle_mod, case):
    import torch.multiprocessing as mp
    world = 3 if "3ranks" in case else 2
    precision = 32 if "fp32" in case else 64
    P = wl.base_params(136, 6, 12, grav=[1e-4, 0.0, -2e-4])
    if "walls" in case:
        P["bc_f"][2] = ["wall", "wall"]; P["bc_g"][2] = ["zeroflux", "zeroflux"]; P["bc_s"][2] = ["dirichlet", "dirichlet"]
        P["bc_T"][2] = [1.0, 0.0]
    init = _random_state(P, 96)
    nsteps = 7
    o = oracle_mod.Oracle(P); o.init(*init); o.step(nsteps)
    ref = o.read_macro(); o.close()
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, P, init, "events" if "events" in case else "flags", precision, nsteps, out))
             for r in range(world)]
    for p in procs:
        p.start()
    try:
        res = dict(out.get(timeout=240) for _ in procs)
        for p in procs:
            p.join(timeout=60)
            assert p.exitcode == 0
    finally:
        for p in procs:
            if p.is_alive():
                p.kill()
    for i, name in enumerate(("phi", "u", "p", "T")):
        got = np.concatenate([res[r][i] for r in range(world)], axis=res[0][i].ndim - 3)
        err = float(np.abs(got.astype(np.float64) - ref[i]).max())
        if precision == 64:
            assert err <= 1e-10, (case, name, err)
        else:
            assert err / max(float(np.abs(ref[i]).max()), 1e-30) <= 1e-4, (case, name, err)
