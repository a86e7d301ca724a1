"""Slab decomposition on ONE GPU (paper_2003_06342_b200/slabs.py, include/lbm.h "slab decomposition"): several slab
contexts in one process, ghost layers handed over with lbm_halo_pack / lbm_halo_unpack between the phases of a step.
The stitched result must equal the undecomposed CUDA run -- BIT FOR BIT when every face is periodic (same kernels, same
neighbour values); to a few ulp when physical faces are present, because a node may then fall into a tile that takes the
boundary instantiation of the kernel in one run and the plain one in the other (the two are compiled separately and
contract multiply-adds differently) -- and the CPU oracle of the whole domain within the fp64 tolerance.  Both schedules are
checked: the overlapped one (boundary layers first, exchanges on a second stream ordered by events, ghost layers not
computed; the default) and the plain one-stream sequence.  No kernel waits on another: the order is the streams'."""
import numpy as np
import pytest

from paper_2003_06342_b200 import slabs
from paper_2003_06342_b200 import workloads as wl
from test_oracle_bruteforce import _random_state

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
ULP64, ULP32 = 1e-14, 2e-6      # slabs against the undecomposed CUDA run when physical faces are present


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2003_06342_b200 import binding
    binding.load_library()
    return binding


def _state(group_or_sim, gpu):
    out = dict(zip(("phi", "u", "p", "T"), group_or_sim.read_macro()))
    for which, name in enumerate("fgs"):
        out[name + "*"] = group_or_sim.read_pops(which, gpu.STAGE_POSTCOLLISION)
        out[name] = group_or_sim.read_pops(which, gpu.STAGE_STREAMED)
    return out


def _check(gpu, oracle_mod, P, init, nslabs_list, horizons, precision=64, oracle=True, exact=True):
    single = gpu.LBM(P, precision)
    single.init(*init)
    # per slab count: overlapped schedule with the ghost layers pushed straight into the neighbour (lbm_halo_push), the plain
    # schedule with pushes, and the overlapped schedule with the buffered pack / unpack exchange a multi-process run uses
    nslabs_list = [n for n in nslabs_list for _ in range(3)]
    groups = [slabs.SlabGroup(P, n, precision, overlap=(i % 3 != 1), push=(i % 3 != 2)) for i, n in enumerate(nslabs_list)]
    for g in groups:
        g.init(*init)
    o = None
    if oracle:
        o = oracle_mod.Oracle(P)
        o.init(*init)
    done = 0
    for h in horizons:
        single.step(h - done)
        for g in groups:
            g.step(h - done)
        if o:
            o.step(h - done)
        done = h
        ref = _state(single, gpu)
        for n, g in zip(nslabs_list, groups):
            got = _state(g, gpu)
            for k, v in ref.items():
                assert got[k].shape == v.shape, (n, k, got[k].shape, v.shape)
                err = np.abs(got[k].astype(np.float64) - v).max()
                ok = np.array_equal(got[k], v) if exact else err <= (ULP64 if precision == 64 else ULP32)
                assert ok, "%d slabs, step %d, %s: max diff %g" % (n, h, k, err)
        if o:
            for a, b, name in zip(groups[-1].read_macro(), o.read_macro(), ("phi", "u", "p", "T")):
                assert np.abs(a - b).max() <= TOL64, (h, name)
            for which in range(3):
                assert np.abs(groups[-1].read_pops(which, gpu.STAGE_STREAMED) - o.read_pops(which)).max() <= TOL64
    single.destroy()
    for g in groups:
        g.destroy()
    if o:
        o.close()


def test_film_3d_walls_in_z(gpu, oracle_mod):
    """Config-4 recipe (walls and heated plate in z): 2 and 3 slabs, ragged split 22 = 8 + 7 + 7."""
    P, st = wl.config4_film3d(40, 24, 22, h0=7.0, amp=2.0)
    _check(gpu, oracle_mod, P, (st["phi"], st["T"], None, None), [2, 3], [1, 2, 9], exact=False)


def test_periodic_box_3d(gpu, oracle_mod):
    """Periodic in z: a single slab is its own neighbour; 2 slabs exchange both sides with the same peer."""
    P = wl.base_params(136, 6, 10, grav=[1e-4, -2e-4, 5e-5])
    _check(gpu, oracle_mod, P, _random_state(P, 61), [1, 2, 5], [1, 6])


def test_d3q15_slabs(gpu, oracle_mod):
    P, st = wl.config4_film3d(40, 24, 14, h0=5.0, amp=1.5, lat_f="D3Q15")
    _check(gpu, oracle_mod, P, (st["phi"], st["T"], None, None), [3], [1, 6], exact=False)


def test_film_2d_cut_along_y(gpu, oracle_mod):
    P, st = wl.config3_film2d(40, 30, h0=8.0, amp=2.0)
    _check(gpu, oracle_mod, P, (st["phi"], st["T"], None, None), [2, 4], [1, 12], exact=False)


def test_periodic_2d_both_lattice_sets(gpu, oracle_mod):
    for lat_s in ("D2Q5", "D2Q9"):
        P = wl.base_params(33, 17, 1, lat_s=lat_s, theta_I=0.05)
        _check(gpu, oracle_mod, P, _random_state(P, 62), [1, 3], [1, 8])


def test_mixed_faces_dirichlet_and_open(gpu, oracle_mod):
    """Physical faces of every kind at the two ends of the cut axis, walls in x as well."""
    P = wl.base_params(24, 12, 9)
    P["bc_f"][2] = ["wall", "open"]; P["bc_g"][2] = ["dirichlet", "zeroflux"]; P["bc_s"][2] = ["zeroflux", "dirichlet"]
    P["bc_phi"][2] = [1.0, 0.0]; P["bc_T"][2] = [0.0, 0.3]; P["bc_p"][2] = [0.0, 1e-3]
    P["bc_f"][0] = ["wall", "wall"]; P["bc_g"][0] = ["zeroflux", "zeroflux"]; P["bc_s"][0] = ["zeroflux", "zeroflux"]
    z = (np.arange(9) + 0.5)[:, None, None]
    phi = 0.5 * (1 - np.tanh(2 * (z - 4.0) / 3.0)) + np.zeros((9, 12, 24))
    rng = np.random.Generator(np.random.PCG64(63))
    phi = phi + 1e-3 * rng.uniform(-1, 1, phi.shape)
    T = 0.1 * rng.uniform(-1, 1, phi.shape)
    _check(gpu, oracle_mod, P, (phi, T, None, None), [3], [1, 5], exact=False)


def test_fp32_slabs(gpu, oracle_mod):
    P, st = wl.config4_film3d(136, 8, 12, h0=5.0, amp=1.0)
    _check(gpu, oracle_mod, P, (st["phi"], st["T"], None, None), [3], [1, 6], precision=32, oracle=False, exact=False)


def test_prescribed_velocity_slabs(gpu, oracle_mod):
    P = wl.base_params(40, 28, 1, prescribed_u=True)
    _check(gpu, oracle_mod, P, _random_state(P, 64), [2], [1, 5])


def test_slab_api_states(gpu):
    P = wl.base_params(16, 8, 6)
    Pl = slabs.local_params(P, 0, 2)
    assert Pl["halo"] == (1, 1)
    import torch
    sim = gpu.LBM(Pl, 64)
    L = gpu.load_library()
    buf = torch.empty(sim.halo_bytes(gpu.HALO_POPS), dtype=torch.uint8, device="cuda")
    assert sim.halo_bytes(gpu.HALO_POPS) == 7 * 16 * 8 * 8             # 5 + 1 + 1 populations of one 16 x 8 layer, fp64
    assert sim.halo_bytes(gpu.HALO_PHI) > 16 * 8 * 8                   # one padded layer
    with pytest.raises(gpu.LBMError):
        sim.halo_pack(gpu.HALO_POPS, 0, buf)                           # before lbm_init
    sim.init(np.full((5, 8, 16), 0.5))
    assert L.lbm_step(sim._h, 1) == -5                                 # slabs step by phases
    with pytest.raises(gpu.LBMError):
        sim.step_phase(1)                                              # phase 0 comes first
    with pytest.raises(gpu.LBMError):
        sim.halo_pack(gpu.HALO_PHI, 0, buf)                            # phi travels between the phases only
    sim.halo_pack(gpu.HALO_POPS, 1, buf)
    sim.step_phase(0)
    with pytest.raises(gpu.LBMError):
        sim.halo_pack(gpu.HALO_POPS, 0, buf)
    with pytest.raises(gpu.LBMError):
        sim.step_phase(0)
    sim.halo_pack(gpu.HALO_PHI, 0, buf)
    sim.halo_unpack(gpu.HALO_PHI, 1, buf)
    sim.step_phase(1, True)
    assert sim.step_count == 1
    sim.destroy()
    # a context without ghost layers refuses the halo calls; a ghost side needs a periodic-kind face
    sim = gpu.LBM(P, 64)
    sim.init(np.full((6, 8, 16), 0.5))
    with pytest.raises(gpu.LBMError):
        sim.halo_bytes(gpu.HALO_PHI)
    sim.destroy()
    Pw, _ = wl.config4_film3d(16, 8, 6)
    Pw["halo"] = (1, 0)                                                # ghost layer on a wall face
    with pytest.raises(gpu.LBMError):
        gpu.LBM(Pw, 64)
    Pm = slabs.local_params(Pw, 0, 2)
    Pm["halo"] = (0, 0)                                                # mixed kinds without the ghost layer
    with pytest.raises(gpu.LBMError):
        gpu.LBM(Pm, 64)


def test_push_to_a_mapped_workspace(gpu, oracle_mod):
    """lbm_halo_push_mapped: the neighbour given by its parameters and the address of its workspace only (the form a peer-mapped
    multi-process run uses) -- same bits as the undecomposed run on a periodic box, walls within a few ulp, oracle within 1e-10."""
    P = wl.base_params(136, 6, 11, grav=[1e-4, -2e-4, 5e-5])
    init = _random_state(P, 67)
    single = gpu.LBM(P, 64); single.init(*init); single.step(7)
    o = oracle_mod.Oracle(P); o.init(*init); o.step(7)
    for n in (2, 3):
        g = slabs.SlabGroup(P, n, 64, overlap=True, push="mapped"); g.init(*init); g.step(7)
        for k, v in _state(single, gpu).items():
            assert np.array_equal(_state(g, gpu)[k], v), (n, k)
        for a, b in zip(g.read_macro(), o.read_macro()):
            assert np.abs(a - b).max() <= TOL64
        g.destroy()
    single.destroy(); o.close()
    P, st = wl.config4_film3d(40, 24, 14, h0=5.0, amp=1.5)
    single = gpu.LBM(P, 32); single.init(st["phi"].astype(np.float32), st["T"].astype(np.float32)); single.step(6)
    g = slabs.SlabGroup(P, 3, 32, overlap=False, push="mapped"); g.init(st["phi"].astype(np.float32), st["T"].astype(np.float32)); g.step(6)
    for a, b in zip(g.read_macro(), single.read_macro()):
        assert np.abs(a.astype(np.float64) - b).max() <= ULP32
    # a neighbour that does not fit: other row length
    bad = dict(g.slabs[1].P, nx=P["nx"] + 2)
    with pytest.raises(gpu.LBMError):
        g.slabs[0].sim.halo_push_mapped(slabs.HALO_POPS, 1, bad, g.slabs[1].sim.workspace_ptr)
    g.destroy(); single.destroy()


def test_graph_replay_of_the_overlapped_step(gpu):
    """Small slabs replay their overlapped step from a CUDA graph of two consecutive steps captured across the compute and the
    exchange stream, one graph per buffer parity (slabs.SlabGroup, lbm_note_replay): same bits as the launches themselves, from
    even and from odd step counts, and the contexts' step counters follow the replays."""
    for P, seed in ((wl.base_params(136, 6, 12, grav=[1e-4, -2e-4, 5e-5]), 65), (wl.base_params(40, 36, 1, grav=[1e-4, -1e-4, 0.0]), 66)):
        init = _random_state(P, seed)
        a = slabs.SlabGroup(P, 3, 64, overlap=True, graph=True)
        b = slabs.SlabGroup(P, 3, 64, overlap=True, graph=False)
        for g in (a, b):
            g.init(*init)
        total = 0
        for n in (1, 12, 11, 9):          # parities 1, 1, 0 at the start of the graph-eligible calls
            a.step(n); b.step(n); total += n
            assert len(a._graphs) >= (1 if total > 1 else 0) and not b._graphs
            assert all(s.sim.step_count == total for s in a.slabs), [s.sim.step_count for s in a.slabs]
            assert [s.sim.launch_count for s in a.slabs] == [s.sim.launch_count for s in b.slabs]
            for x, y in zip(_state(a, gpu).values(), _state(b, gpu).values()):
                assert np.array_equal(x, y), (n, total)
        assert len(a._graphs) == 2
        a.destroy(); b.destroy()
