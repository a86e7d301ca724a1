"""lbm_read_pops_noalloc (include/lbm.h): the streamed populations through the static device scratch instead of a temporary
from cudaMalloc, against the existing lbm_read_pops.  Collected last on purpose (file name): the suite runs with pytest -x.
Passes alone in a fresh process and after the other tests (it depends on nothing but its own contexts)."""
import numpy as np
import pytest

from paper_2003_06342_b200 import workloads as wl
from test_oracle_bruteforce import _random_state

pytestmark = pytest.mark.gpu
TOL64 = 1e-10   # the fp64 parity bar of tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_06342_b200 import binding
    binding.load_library()
    return binding


def test_read_pops_noalloc_matches_read_pops_twice_in_a_row(gpu):
    # two contexts, two calls in a row on each, all three lattices, both stages; the second call reuses the scratch the first
    # one (and the other context, with a different size) left behind
    P3 = wl.base_params(40, 10, 7, grav=[1e-4, 0.0, -2e-4])
    P3["bc_f"][2] = ["wall", "wall"]; P3["bc_g"][2] = ["zeroflux", "zeroflux"]; P3["bc_s"][2] = ["dirichlet", "dirichlet"]
    P3["bc_T"][2] = [1.0, 0.0]
    P2 = wl.base_params(33, 17, 1, lat_s="D2Q9", grav=[0.0, -1e-4, 0.0])
    sims = []
    for P, seed, prec in ((P3, 91, 64), (P2, 92, 32)):
        sim = gpu.LBM(P, prec)
        sim.init(*[a.astype(sim.dtype) for a in _random_state(P, seed)])
        sims.append(sim)
    for steps in (3, 2):                       # call 1 after 3 steps, call 2 after 5
        for sim in sims:
            sim.step(steps)
            for which in (gpu.POPS_F, gpu.POPS_G, gpu.POPS_S):
                for stage in (gpu.STAGE_STREAMED, gpu.STAGE_POSTCOLLISION):
                    want = sim.read_pops(which, stage)
                    got = sim.read_pops_noalloc(which, stage)
                    assert got.shape == want.shape and np.isfinite(got).all()
                    assert float(np.abs(got - want).max()) <= TOL64, (which, stage)
    for sim in sims:
        sim.destroy()


def test_read_pops_noalloc_rejects_what_does_not_fit(gpu):
    P = wl.base_params(64, 64, 32)             # D3Q19 in double: 19 * 131072 * 8 B = 19.9 MB > 8 MiB
    sim = gpu.LBM(P, 64)
    sim.init(np.full((32, 64, 64), 0.5))
    sim.step(1)
    L = gpu.load_library()
    out = np.empty((19, 32, 64, 64))
    rc = L.lbm_read_pops_noalloc(sim._h, gpu.POPS_F, gpu.STAGE_STREAMED, out.ctypes.data)
    assert rc == -7 and "scratch" in gpu.lbm_strerror(rc)
    with pytest.raises(gpu.LBMError):
        sim.read_pops_noalloc(gpu.POPS_F)
    # D3Q7 in double on the same grid fits: 7 * 131072 * 8 B = 7.3 MB
    assert np.array_equal(sim.read_pops_noalloc(gpu.POPS_S), sim.read_pops(gpu.POPS_S))
    # before the first step there are no streamed populations, as for lbm_read_pops
    sim.init(np.full((32, 64, 64), 0.5))
    assert L.lbm_read_pops_noalloc(sim._h, gpu.POPS_S, gpu.STAGE_STREAMED, out.ctypes.data) == -5
    assert L.lbm_read_pops_noalloc(sim._h, 7, gpu.STAGE_STREAMED, out.ctypes.data) == -1
    sim.destroy()
