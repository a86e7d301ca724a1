"""Memory-safety checks of our own over tests/sanitizer_cases.py, standing in for compute-sanitizer where that tool is closed
(profiles/r2_sanitizer.md):

* guard bands: the workspace lent to the library sits between two 1 MiB bands of a known byte; after init, steps and every read
  call the bands must be untouched (an out-of-range store of any kernel would land there or fault);
* poison: the workspace starts as all-ones bytes (NaN in both precisions), so a kernel that reads an element nobody wrote
  (an uninitialised ghost image, a stale buffer) produces NaN in the outputs, which are checked finite and, in fp64, against
  the oracle;
* determinism: the same case run twice gives the same bits (a shared-memory or hand-over race between threads would, sooner or
  later, not).
"""
import numpy as np
import pytest

from sanitizer_cases import cases
from test_oracle_bruteforce import _random_state

pytestmark = pytest.mark.gpu
GUARD = 1 << 20
BAND = 0xA5


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_06342_b200 import binding
    binding.load_library()
    return binding


def _guarded(gpu, P, prec):
    import torch
    n = gpu.lbm_workspace_bytes(P, prec)
    raw = torch.empty(n + 2 * GUARD, dtype=torch.uint8, device="cuda")
    raw[:GUARD] = BAND
    raw[GUARD + n:] = BAND
    raw[GUARD:GUARD + n] = 0xFF
    return raw, raw[GUARD:GUARD + n]


def _bands_ok(raw, n):
    return bool((raw[:GUARD] == BAND).all()) and bool((raw[GUARD + n:] == BAND).all())


@pytest.mark.parametrize("prec", [64, 32])
def test_guard_bands_poison_and_determinism(gpu, oracle_mod, prec):
    for name, P, seed in cases():
        init = _random_state(P, seed)
        ref = None
        if prec == 64:
            o = oracle_mod.Oracle(P); o.init(*init); o.step(7)
            ref = o.read_macro(); o.close()
        for kernels in ((), ("pops_gather",), ("pops_staged",), ("phi_ldg",), ("no_graph", "no_pdl"), ("one_node",),
                        ("one_node", "pops_staged")):   # fp32 3D: the first three run pairs of nodes, the last two one node per thread
            Q = dict(P); Q["kernels"] = kernels
            runs = []
            for rep in range(2):
                raw, ws = _guarded(gpu, Q, prec)
                sim = gpu.LBM(Q, prec, workspace=ws)
                sim.init(*[a.astype(sim.dtype) for a in init])
                sim.step(7)
                out = list(sim.read_macro())
                for w in range(3):
                    out.append(sim.read_pops(w, gpu.STAGE_STREAMED))
                    out.append(sim.read_pops(w, gpu.STAGE_POSTCOLLISION))
                sim.sync()
                assert _bands_ok(raw, ws.numel()), (name, prec, kernels, "store outside the workspace")
                assert all(np.isfinite(a).all() for a in out), (name, prec, kernels, "read of an element nobody wrote")
                sim.destroy()
                runs.append(out)
            for a, b in zip(*runs):
                assert np.array_equal(a, b), (name, prec, kernels, "two runs differ")
            if ref is not None:
                for a, b, f in zip(runs[0][:4], ref, ("phi", "u", "p", "T")):
                    assert float(np.abs(a - b).max()) <= 1e-10, (name, kernels, f)
