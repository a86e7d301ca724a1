"""Pin P18: the C oracle against the independent NumPy transcription (tests/np_bruteforce.py) on tiny grids,
all boundary kinds, 2D and 3D, >= 10 steps, compared element by element on macros and populations."""
import numpy as np
import pytest

from np_bruteforce import NPModel
from paper_2003_06342_b200 import workloads as wl

TOL = 1e-13


def _random_state(P, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = (P["nz"], P["ny"], P["nx"])
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    # a diffuse blob (so that gradients, normals and curvature are all non-trivial) plus noise
    r = np.sqrt((x - nx / 2.3) ** 2 + (y - ny / 1.9) ** 2 + ((z - nz / 2.1) ** 2 if nz > 1 else 0))
    phi = 0.5 * (1 + np.tanh(2 * (r - 0.3 * min(nx, ny)) / 2.0)) + 0.01 * rng.uniform(-1, 1, shape)
    T = P["T_sat"] + rng.uniform(-0.5, 0.5, shape)
    u = 0.02 * rng.uniform(-1, 1, (3,) + shape)
    if nz == 1:
        u[2] = 0
    p = 0.01 * rng.uniform(-1, 1, shape)
    return phi, T, u, p


def _compare(oracle_mod, P, steps, seed, TOL=TOL):
    phi, T, u, p = _random_state(P, seed)
    o = oracle_mod.Oracle(P)
    o.init(phi, T, u, p)
    m = NPModel(P)
    m.init(phi, T, u, p)
    for chunk in (1, steps - 1):
        o.step(chunk)
        m.step(chunk)
        ophi, ou, op, oT = o.read_macro()
        assert np.abs(ophi - m.phi).max() < TOL
        assert np.abs(ou - m.u).max() < TOL
        assert np.abs(op - m.p).max() < TOL
        assert np.abs(oT - m.T).max() < TOL
        for which, key in enumerate("fgs"):
            e_o, _, _ = oracle_mod.lattice(P["lat_" + key])
            pops_o = o.read_pops(which, oracle_mod.POPS_STREAMED)
            vec = m.vectors(key)
            for i, v in enumerate(e_o):
                j = int(np.where((vec == v).all(axis=1))[0][0])
                assert np.abs(pops_o[i] - m.pops[key][j]).max() < TOL, (key, i)
    o.close()


def test_2d_periodic(oracle_mod):
    P = wl.base_params(8, 8, 1, grav=[1e-4, -2e-4, 0.0], nu_l=0.05, nu_g=0.2, force=[2e-5, 1e-5, 0.0])
    _compare(oracle_mod, P, 12, 11)


def test_physical_units_dx_dt_not_one(oracle_mod):
    """dx = 0.5, dt = 0.2 (c = 2.5): every place where c, c_s^2 = e^2 c^2, 1/dx, 1/dx^2 or dt enters (PAPER.md:190, 208, 236, 272,
    Eq.35-36) must agree between the two transcriptions; the paper's own runs are in physical units."""
    P = wl.base_params(8, 8, 1, dx=0.5, dt=0.2, grav=[1e-3, -2e-3, 0.0], force=[2e-4, 1e-4, 0.0], W=2.0)
    P["bc_f"][1] = ["wall", "wall"]; P["bc_g"][1] = ["zeroflux", "dirichlet"]; P["bc_s"][1] = ["dirichlet", "zeroflux"]
    P["bc_phi"][1] = [0.0, 1.0]; P["bc_T"][1] = [0.7, 0.0]
    _compare(oracle_mod, P, 12, 91)
    _compare(oracle_mod, wl.base_params(8, 8, 8, dx=0.5, dt=0.2, grav=[1e-3, 0.0, -2e-3], W=2.0), 12, 92)


def test_2d_periodic_d2q9_heat(oracle_mod):
    P = wl.base_params(8, 8, 1, lat_s="D2Q9", theta_I=0.05)
    _compare(oracle_mod, P, 12, 12)


def test_2d_walls_dirichlet(oracle_mod):
    P = wl.base_params(8, 8, 1, grav=[0.0, -1e-4, 0.0])
    P["bc_f"][1] = ["wall", "wall"]
    P["bc_g"][1] = ["zeroflux", "dirichlet"]
    P["bc_s"][1] = ["dirichlet", "zeroflux"]
    P["bc_phi"][1] = [0.0, 1.0]
    P["bc_T"][1] = [0.7, 0.0]
    _compare(oracle_mod, P, 12, 13)


def test_2d_open_face_and_x_walls(oracle_mod):
    P = wl.base_params(10, 6, 1)
    P["bc_f"][0] = ["wall", "open"]
    P["bc_g"][0] = ["dirichlet", "dirichlet"]
    P["bc_s"][0] = ["dirichlet", "dirichlet"]
    P["bc_phi"][0] = [1.0, 0.0]
    P["bc_T"][0] = [1.0, 0.0]
    P["bc_p"][0] = [0.0, 0.003]
    _compare(oracle_mod, P, 12, 14)


def test_2d_two_nonperiodic_axes(oracle_mod):
    P = wl.base_params(8, 7, 1)
    for a in (0, 1):
        P["bc_f"][a] = ["wall", "wall"]
        P["bc_g"][a] = ["dirichlet", "zeroflux"]
        P["bc_s"][a] = ["zeroflux", "dirichlet"]
        P["bc_phi"][a] = [0.9 - 0.1 * a, 0.0]
        P["bc_T"][a] = [0.0, 0.4 - 0.1 * a]
    # corner links (two non-periodic faces crossed: lowest axis decides, S8-v) make a violent little flow
    # that amplifies round-off; the first steps agree to 1e-16, so a looser bound still catches any rule mismatch
    _compare(oracle_mod, P, 10, 15, TOL=1e-11)


def test_3d_periodic(oracle_mod):
    P = wl.base_params(8, 8, 8, grav=[1e-4, 0.0, -2e-4], nu_l=0.2, nu_g=0.04, force=[0.0, 1e-5, -2e-5])
    _compare(oracle_mod, P, 10, 16)


def test_3d_walls_z(oracle_mod):
    P = wl.base_params(8, 6, 7, grav=[0.0, 0.0, -1e-4])
    P["bc_f"][2] = ["wall", "wall"]
    P["bc_g"][2] = ["zeroflux", "zeroflux"]
    P["bc_s"][2] = ["dirichlet", "dirichlet"]
    P["bc_T"][2] = [1.0, 0.0]
    _compare(oracle_mod, P, 10, 17)


def test_2d_prescribed_velocity(oracle_mod):
    P = wl.base_params(8, 8, 1, prescribed_u=True, nu_l=0.05, nu_g=0.2)
    _compare(oracle_mod, P, 10, 19)


def test_3d_d3q15_navier_stokes_lattice(oracle_mod):
    P = wl.base_params(6, 7, 8, lat_f="D3Q15", grav=[1e-4, -2e-4, 5e-5])
    _compare(oracle_mod, P, 10, 20)
    P = wl.base_params(8, 6, 7, lat_f="D3Q15", grav=[0.0, 0.0, -1e-4])
    P["bc_f"][2] = ["wall", "wall"]; P["bc_g"][2] = ["zeroflux", "zeroflux"]; P["bc_s"][2] = ["dirichlet", "dirichlet"]
    P["bc_T"][2] = [1.0, 0.0]
    _compare(oracle_mod, P, 8, 21)


def test_3d_flags_off(oracle_mod):
    P = wl.base_params(6, 8, 6, phase_change=False, latent_heat=False)
    _compare(oracle_mod, P, 10, 18)


@pytest.mark.parametrize("name", ["D2Q5", "D2Q9", "D3Q7", "D3Q19", "D3Q15"])
def test_lattice_tables(oracle_mod, name):
    """Weights sum to 1, first moment 0, second moment e2 * identity, opposite pairs present; the typed
    tables of the oracle equal the generated shells of the NumPy model as sets."""
    from np_bruteforce import make_lattice
    e, w, e2 = oracle_mod.lattice(name)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs((w[:, None] * e).sum(axis=0)).max() < 1e-16
    dim = 2 if name.startswith("D2") else 3
    m2 = np.einsum("i,ia,ib->ab", w, e.astype(float), e.astype(float))
    assert np.abs(m2[:dim, :dim] - e2 * np.eye(dim)).max() < 1e-15
    e_n, w_n, e2_n = make_lattice(name)
    assert abs(e2 - e2_n) < 1e-15
    assert {tuple(v) + (round(ww, 12),) for v, ww in zip(e, w)} == {tuple(v) + (round(ww, 12),) for v, ww in zip(e_n, w_n)}
    assert abs(e2 - {"D2Q5": 1 / 3, "D2Q9": 1 / 3, "D3Q7": 1 / 4, "D3Q19": 1 / 3, "D3Q15": 1 / 3}[name]) < 1e-15
    if name in ("D2Q9", "D3Q19", "D3Q15"):     # Navier-Stokes lattices: isotropic fourth moment e2^2 (dd + dd + dd)
        m4 = np.einsum("i,ia,ib,ic,id->abcd", w, *(e.astype(float),) * 4)
        d = np.eye(3)
        iso = e2 * e2 * (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d) + np.einsum("ad,bc->abcd", d, d))
        assert np.abs(m4[:dim, :dim, :dim, :dim] - iso[:dim, :dim, :dim, :dim]).max() < 1e-15
    if name == "D3Q15":                         # the two direction vectors the paper prints
        assert tuple(e[7]) == (1, 1, 1) and tuple(e[8]) == (-1, 1, 1) and tuple(e[14]) == (1, -1, -1)
