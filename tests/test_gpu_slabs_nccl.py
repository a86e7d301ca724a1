"""DistSlab over NCCL on two GPUs (one process per GPU) against the whole-domain oracle -- periodic and walled slab axis, both
schedules.  Needs two devices: SKIPPED on the one-GPU boxes this repository has been developed and judged on, i.e. the slab path
has never run on more than one GPU (DESIGN.md "Multi-GPU" says so next to every slab claim); the host logic and the message
order are covered on CPU by tests/test_slabs_host.py (gloo, world sizes 2 and 3)."""
import os
import socket

import numpy as np
import pytest

from paper_2003_06342_b200 import workloads as wl
from test_oracle_bruteforce import _random_state

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, P, init, overlap, nsteps, out):
    import torch
    import torch.distributed as dist
    from paper_2003_06342_b200 import slabs
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world)
    sim = slabs.DistSlab(P, rank, world, 64, overlap=overlap)
    sim.init(*init)
    sim.step(nsteps)
    out.put((rank, [np.asarray(a) for a in sim.read_macro()]))
    dist.barrier()
    sim.destroy()
    dist.destroy_process_group()


@pytest.mark.parametrize("overlap", [True, False])
@pytest.mark.parametrize("walls", [False, True])
def test_dist_slab_two_gpus_against_oracle(oracle_mod, overlap, walls):
    import torch
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (the slab path is unmeasured on hardware with more than one)")
    P = wl.base_params(40, 10, 12, grav=[1e-4, 0.0, -2e-4])
    if walls:
        P["bc_f"][2] = ["wall", "wall"]; P["bc_g"][2] = ["zeroflux", "zeroflux"]; P["bc_s"][2] = ["dirichlet", "dirichlet"]
        P["bc_T"][2] = [1.0, 0.0]
    init = _random_state(P, 95)
    o = oracle_mod.Oracle(P); o.init(*init); o.step(6)
    ref = o.read_macro(); o.close()
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, P, init, overlap, 6, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(out.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for i, name in enumerate(("phi", "u", "p", "T")):
        got = np.concatenate([res[0][i], res[1][i]], axis=res[0][i].ndim - 3)
        assert float(np.abs(got - ref[i]).max()) <= 1e-10, name
