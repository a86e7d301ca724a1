"""Small runs of every default kernel for compute-sanitizer: both precisions, 2D and 3D, wide / mid / narrow
tiles, walls and periodic faces, the plainer kernel variants, the CUDA-graph replay and a pair of slabs.

    compute-sanitizer --tool memcheck|racecheck|synccheck|initcheck python tests/sanitizer_cases.py

ONE tool per invocation (and per gpurun call: B200_PROFILING.md).  Prints "sanitizer cases ok" and exits 0 when every case ran
and stayed finite; the sanitizer's own verdict is its "ERROR SUMMARY" line.  Driven by tests/test_gpu_sanitizer.py.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from paper_2003_06342_b200 import binding, slabs, workloads as wl  # noqa: E402
from test_oracle_bruteforce import _random_state  # noqa: E402


def cases():
    P = wl.base_params(250, 6, 5, grav=[1e-4, 0.0, -2e-4])                    # 3D wide tiles (128 + 122), ragged x
    yield "3d wide periodic", P, 11
    P = wl.base_params(64, 5, 6, grav=[0.0, 0.0, -1e-4])                      # 3D 64 x 2 tiles, z walls
    P["bc_f"][2] = ["wall", "wall"]; P["bc_g"][2] = ["zeroflux", "zeroflux"]; P["bc_s"][2] = ["dirichlet", "dirichlet"]
    P["bc_T"][2] = [1.0, 0.0]
    yield "3d mid z walls", P, 12
    P = wl.base_params(20, 9, 7, lat_f="D3Q15")                               # 3D narrow tiles, box with an open face
    for a in range(3):
        P["bc_f"][a] = ["wall", "open" if a == 0 else "wall"]; P["bc_g"][a] = ["dirichlet", "zeroflux"]
        P["bc_s"][a] = ["dirichlet", "zeroflux"]; P["bc_phi"][a] = [0.9, 0.0]; P["bc_T"][a] = [0.2, 0.0]
    yield "3d narrow box D3Q15", P, 13
    P = wl.base_params(140, 12, 1, grav=[1e-4, -1e-4, 0.0], lat_s="D2Q9")     # 2D wide tiles, three D2Q9
    yield "2d wide periodic", P, 14
    P = wl.base_params(40, 20, 1, grav=[0.0, -1e-4, 0.0])                     # 2D narrow tiles, y walls
    P["bc_f"][1] = ["wall", "wall"]; P["bc_g"][1] = ["zeroflux", "dirichlet"]; P["bc_s"][1] = ["dirichlet", "zeroflux"]
    P["bc_phi"][1] = [0.0, 1.0]; P["bc_T"][1] = [0.7, 0.0]
    yield "2d narrow y walls", P, 15


def main():
    n = 0
    for name, P, seed in cases():
        init = _random_state(P, seed)
        for prec in (64, 32):
            for kernels in ((), ("pops_gather",), ("pops_staged",), ("phi_ldg",), ("no_graph", "no_pdl"), ("one_node",),
                            ("one_node", "pops_staged")):
                Q = dict(P); Q["kernels"] = kernels
                sim = binding.LBM(Q, prec)
                sim.init(*[a.astype(sim.dtype) for a in init])
                sim.step(7)                       # small grids: plain steps, graph capture, replay, macro step
                out = sim.read_macro()
                for w in range(3):
                    sim.read_pops(w, binding.STAGE_STREAMED)
                    sim.read_pops_noalloc(w, binding.STAGE_STREAMED)
                assert all(np.isfinite(a).all() for a in out), (name, prec, kernels)
                sim.destroy()
                n += 1
    P = wl.base_params(64, 6, 9, grav=[0.0, 0.0, -1e-4])                      # two slabs, ghost-layer exchange
    P["bc_f"][2] = ["wall", "wall"]; P["bc_g"][2] = ["zeroflux", "zeroflux"]; P["bc_s"][2] = ["dirichlet", "dirichlet"]
    P["bc_T"][2] = [1.0, 0.0]
    for prec in (64, 32):
        grp = slabs.SlabGroup(P, 2, prec)
        grp.init(*[a.astype(np.float64 if prec == 64 else np.float32) for a in _random_state(P, 16)])
        grp.step(4)
        assert np.isfinite(grp.read_macro()[0]).all()
        grp.destroy()
        n += 1
    print("sanitizer cases ok: %d contexts" % n)


if __name__ == "__main__":
    main()
