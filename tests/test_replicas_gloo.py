"""N > 1 path on CPU: the replica plumbing of bench.py (barrier, max-over-ranks time, summed units) on the gloo
backend with world_size 2.  The data path has no collective ("replicas only"), so this is all there is to cover."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2003_06342_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    r, lr, w = replicas.init_process_group("gloo")
    assert (r, lr, w) == (rank, rank, world)
    replicas.barrier()
    ms_local = 10.0 + 5.0 * rank            # rank 1 is the slow one
    ms, units = replicas.reduce_job(ms_local, 1000.0 * (rank + 1))
    seed = replicas.replica_seed(4, rank)
    out.put((rank, ms, units, seed))
    replicas.barrier()
    dist.destroy_process_group()


def test_two_replicas_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]          # max over ranks, seen by every rank
    assert [r[2] for r in res] == [3000.0, 3000.0]      # units summed over ranks
    assert res[0][3] != res[1][3]                       # replicas are seeded differently
    assert abs(replicas.job_throughput_mlups(15.0, 3000.0e6) - 3000.0 / 0.015) < 1e-6


def test_single_process_passthrough():
    assert replicas.env_rank()[2] >= 1
    assert replicas.reduce_job(3.0, 7.0) == (3.0, 7.0)
