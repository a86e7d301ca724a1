"""Multi-GPU plumbing: independent replicas, one process per GPU ("replicas only").

The path is defined on one GPU (north_star: no sharding, no inter-GPU communication), so ``bench.py --gpus N`` runs
N independent copies of the workload, each seeded by its rank, with no data-path collective.  ``torch.distributed``
is used for the start/stop barriers and for the max-over-ranks reduction of the device time only.  The same helpers
run on the ``gloo`` backend on CPU (tests/test_replicas_gloo.py).
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when launched directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init_process_group(backend: str):
    """Join the job's process group when WORLD_SIZE > 1 (MASTER_ADDR/MASTER_PORT from the environment)."""
    import torch.distributed as dist
    rank, local_rank, world = env_rank()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica gets its own seeded input (same recipe, different random numbers)."""
    return int(base_seed) + 1000 * int(rank)


def reduce_job(ms_local: float, units_local: float, device=None):
    """Whole-job numbers from per-rank ones: (max over ranks of the elapsed ms, sum over ranks of the units)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(ms_local), float(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def job_throughput_mlups(ms_job: float, lattice_updates_job: float) -> float:
    """MLUPS = lattice updates / (1e6 * seconds)."""
    return lattice_updates_job / (ms_job * 1e-3) / 1e6
