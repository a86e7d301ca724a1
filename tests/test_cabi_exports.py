"""Host-side checks of the C-ABI library that need no GPU: it builds for sm_100a, loads, exports every symbol that
include/lbm.h declares, sizes workspaces, validates parameters and refuses to run without a device."""
import ctypes as C
import os
import re

import pytest

from paper_2003_06342_b200 import binding, build, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "lbm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_functions()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_sass_is_sm100a(lib):
    out = os.popen("cuobjdump -lelf %s 2>/dev/null" % binding.LIB_PATH).read()
    assert "sm_100a" in out


def test_sass_has_tma_and_async_copies(lib):
    """The Blackwell-native staging must really be in the shipped binary (B200_PROFILING.md "What proves a Blackwell-native
    kernel"): UTMALDG = the phi halo box by cp.async.bulk.tensor, SYNCS = its mbarrier, LDGSTS = the per-thread cp.async of the
    populations.  A regression to plain loads would pass every parity test; this one fails."""
    sass = os.popen("cuobjdump -sass %s 2>/dev/null" % binding.LIB_PATH).read()
    assert sass.count("UTMALDG") >= 16 and sass.count("SYNCS.PHASECHK") >= 16 and sass.count("LDGSTS") >= 100
    # per kernel family: the default K_main of every lattice set and precision carries all three
    funcs = sass.split("Function : ")[1:]
    smem = [f for f in funcs if f.startswith("_ZN3lbm11k_main_smem")]
    assert len(smem) >= 16
    for f in smem:
        assert "UTMALDG" in f and "LDGSTS" in f and "SYNCS" in f, f[:200]
    phitma = [f for f in funcs if f.startswith("_ZN3lbm13k_main_phitma")]
    assert phitma and all("UTMALDG" in f for f in phitma)
    # fp32 3D: two nodes per thread -- the packed f32x2 arithmetic of sm_100 and the staged pair copies (k_main_pair.cuh)
    pair = [f for f in funcs if f.startswith("_ZN3lbm16k_main_pair_smem")]
    assert len(pair) >= 4
    for f in pair:
        assert f.count("FFMA2") >= 50 and f.count("FADD2") >= 50 and "UTMALDG" in f and "LDGSTS" in f, f[:200]
    kphi_pair = [f for f in funcs if f.startswith("_ZN3lbm10k_phi_pair")]
    assert kphi_pair and all(f.count("FADD2") >= 30 for f in kphi_pair)


def test_workspace_bytes_accounting(lib):
    P, _ = wl.config4_film3d(nx=8, ny=8, nz=8)      # parameters only matter
    P.update(nx=256, ny=256, nz=512)
    n = 256 * 256 * 512
    b64 = binding.lbm_workspace_bytes(P, 64)
    # two buffers of 19+7+7 populations + 2 Pdot, u(3), p, T, scratch + two padded phi
    lower = (2 * 33 + 8) * n * 8 + 2 * 258 * 258 * 514 * 8
    assert lower <= b64 <= lower * 1.001
    b32 = binding.lbm_workspace_bytes(P, 32)
    # float populations, Pdot, macros, scratch; the two padded phi arrays stay double (include/lbm.h "Precisions")
    lower32 = (2 * 33 + 8) * n * 4 + 2 * 258 * 258 * 514 * 8
    assert lower32 <= b32 <= lower32 * 1.001
    assert b64 < 180e9


def test_parameter_validation(lib):
    P = wl.base_params(16, 16, 1)
    assert binding.lbm_workspace_bytes(P) > 0
    bad = dict(P, lat_f="D3Q19")                   # 3D lattice on a 2D grid
    assert binding.lbm_workspace_bytes(bad) == 0
    bad = dict(P, W=0.0)
    assert binding.lbm_workspace_bytes(bad) == 0
    bad = wl.base_params(16, 16, 1)
    bad["bc_f"][1] = ["wall", "periodic"]          # unpaired periodic face
    assert binding.lbm_workspace_bytes(bad) == 0
    bad = wl.base_params(16, 16, 1)
    bad["bc_f"][1] = ["wall", "wall"]              # f non-periodic but g, s periodic on that axis
    assert binding.lbm_workspace_bytes(bad) == 0
    bad = wl.base_params(16, 16, 1, lat_g="D2Q5")  # lattice set not built
    assert binding.lbm_workspace_bytes(bad) == 0
    assert binding.lbm_workspace_bytes(P, precision=16) == 0


def test_strerror_and_null_safety(lib):
    assert binding.lbm_strerror(0) == "ok"
    assert "state" in binding.lbm_strerror(-5)
    lib.lbm_destroy(None)
    assert lib.lbm_step(None, 1) == -1
    assert lib.lbm_step_count(None) == -1


def test_no_cpu_fallback_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    P = wl.base_params(16, 16, 1)
    with pytest.raises(binding.LBMError):
        binding.LBM(P)
    # the raw C call refuses as well: no device, or a host pointer as workspace
    s = binding.make_params(P, 64)
    buf = (C.c_char * (1 << 22))()
    h = C.c_void_p()
    addr = (C.addressof(buf) + 255) // 256 * 256
    rc = lib.lbm_create(C.byref(s), C.c_void_p(addr), 1 << 21, None, C.byref(h))
    assert rc < 0 and not h.value
