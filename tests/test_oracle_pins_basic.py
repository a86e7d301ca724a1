"""Pins of the CPU oracle against what the paper and the mathematics fix -- cheap ones.

T0  harness maths: Stefan roots printed in the paper, script-A integrals, film-boiling numbers.
P5  sigma, W <-> K, H.    P14 identities of the NS source.   P15 uniform fixed point.
P16 stencil exactness / order.   P17 symmetries.   P1 mass conservation.   P3 CAC form equivalence.
"""
import math
import os

import numpy as np
import pytest
from scipy.integrate import quad

import analytic
from paper_2003_06342_b200 import workloads as wl

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])


# ---------------------------------------------------------------- T0: harness maths vs printed numbers
def test_stefan_roots_printed_in_paper():
    """PAPER.md:498, 500; also decides reading G5 of the garbled right-hand side of Eq.(41d)."""
    assert abs(analytic.stefan_xi_two_phase(-0.3, 0.3, 0.0, 0.14, 0.14) - GOLD["stefan_xi_equal_alpha"]) < 2e-6
    for ratio, key in ((10, "stefan_xi_ratio10"), (5, "stefan_xi_ratio5"), (2, "stefan_xi_ratio2")):
        xi = analytic.stefan_xi_two_phase(-0.3, 0.3, 0.05, 1.0, 1.0 / ratio)
        assert abs(xi - GOLD[key]) < 2e-6, (ratio, xi)
        # the RHS exactly as printed does NOT reproduce the printed roots when theta_I != 0
        assert abs(analytic.stefan_xi_printed_rhs(-0.3, 0.3, 0.05, 1.0, 1.0 / ratio) - GOLD[key]) > 1e-2
    assert abs(analytic.stefan_xi_printed_rhs(-0.3, 0.3, 0.0, 1.0, 1.0) - GOLD["stefan_xi_equal_alpha"]) < 2e-6


def test_one_phase_stefan_root():
    assert abs(analytic.stefan_xi_one_phase(0.1) - wl.XI_STEFAN_ST01) < 1e-6


def test_script_A_integrals():
    """Eq.(B.1)-(B.5), W = 2 sqrt 2."""
    W = 2 * math.sqrt(2)
    phi0 = lambda z: 0.5 * (1 + math.tanh(2 * z / W))
    dphi0 = lambda z: (4 / W) * phi0(z) * (1 - phi0(z))
    pphi = lambda z: phi0(z) * (1 - phi0(z))
    I = quad(lambda z: dphi0(z) ** 2, -40, 40)[0]
    J = quad(lambda z: dphi0(z) * pphi(z), -40, 40)[0]
    inner = lambda z: quad(phi0, 0, z)[0]
    G = quad(lambda z: dphi0(z) * pphi(z) * inner(z), -40, 40)[0]
    U = quad(phi0, -60, 0)[0]
    assert abs(I - 1 / (3 * math.sqrt(2))) < 1e-9
    assert abs(J - 1 / 6) < 1e-9
    assert abs(G + (12 * math.log(2) - 10) / (72 * math.sqrt(2))) < 1e-8
    assert abs(U - math.log(2) / math.sqrt(2)) < 1e-9
    A = (G + J * U) / (2 * I)
    assert abs(A - 10 / 48) < 1e-8
    assert abs(A - GOLD["A_coeff"]) < 1e-5
    assert wl.base_params(4, 4)["A"] == 10 / 48


def test_film_boiling_numbers():
    """Table 2 and PAPER.md:531-535."""
    n = analytic.film_boiling_numbers(1.658, 1.0, 5e-4, 2.5e-3, 5e-3, 4.0, 0.025)
    for k in ("lambda_s", "lambda_c", "t_s", "Gr", "Pr", "Ja"):
        assert abs(n[k] - GOLD[k]) <= 1e-3 * abs(GOLD[k]), (k, n[k])


def test_sigma_W_K_H():
    """P5: Eq.(15a) inverted by Eq.(15b); K int (d phi0)^2 = sigma for the profile Eq.(7)."""
    sigma, W = 1e-3, 4.0
    K, H = 1.5 * W * sigma, 12 * sigma / W
    assert abs(math.sqrt(2 * K * H) / 6 - sigma) < 1e-18
    assert abs(math.sqrt(8 * K / H) - W) < 1e-14
    phi0 = lambda z: 0.5 * (1 + math.tanh(2 * z / W))
    e = quad(lambda z: K * ((4 / W) * phi0(z) * (1 - phi0(z))) ** 2, -80, 80)[0]
    assert abs(e - sigma) < 1e-12


# ---------------------------------------------------------------- P15 uniform fixed point
@pytest.mark.parametrize("dims", [(8, 8, 1), (6, 6, 6)])
def test_uniform_state_is_fixed_point(oracle_mod, dims):
    P = wl.base_params(*dims, grav=[0.0, -1e-3, 0.0])
    shape = dims[::-1]
    for phi_val in (0.0, 1.0):  # pure liquid under gravity stays at rest (F_v = 0 in liquid, G6); pure gas: uniform force
        o = oracle_mod.Oracle(P)
        o.init(np.full(shape, phi_val), np.full(shape, P["T_sat"]))
        o.step(5)
        phi, u, p, T = o.read_macro()
        if phi_val == 0.0:   # bit-exact rest state
            assert np.all(phi == 0.0) and np.all(T == P["T_sat"]) and np.all(u == 0.0) and np.all(p == 0.0)
        else:                # uniform free fall of the whole periodic box: phi, T stay uniform to round-off
            assert np.abs(phi - 1.0).max() < 1e-14 and np.abs(T - P["T_sat"]).max() < 1e-14
            assert np.abs(u[1] - u[1].mean()).max() < 1e-16 and u[1].mean() > 0  # gas pushed against g
        o.close()


# ---------------------------------------------------------------- P16 stencils
@pytest.mark.parametrize("dims", [(12, 10, 1), (10, 8, 9)])
def test_stencils_exact_on_quadratics(oracle_mod, dims):
    """Eq.(35),(36) are exact on quadratic polynomials (interior nodes; zero-flux walls so no wrap jump)."""
    P = wl.base_params(*dims, phase_change=False, latent_heat=False)
    for a in range(3 if dims[2] > 1 else 2):
        P["bc_f"][a] = ["wall", "wall"]; P["bc_g"][a] = ["zeroflux", "zeroflux"]; P["bc_s"][a] = ["zeroflux", "zeroflux"]
    nz, ny, nx = dims[::-1]
    z, y, x = np.meshgrid(np.arange(nz) + .5, np.arange(ny) + .5, np.arange(nx) + .5, indexing="ij")
    c = [0.3, -0.2, 0.15, 0.01, -0.02, 0.005, 0.007, -0.004, 0.003]
    if nz == 1:
        z = 0 * z
    phi = c[0] * x + c[1] * y + c[2] * z + c[3] * x * x + c[4] * y * y + c[5] * z * z + c[6] * x * y + c[7] * x * z + c[8] * y * z
    o = oracle_mod.Oracle(P)
    o.init(phi)
    grad, lap, _, _ = o.read_aux()
    sl = (slice(1, -1) if nz > 1 else slice(None), slice(1, -1), slice(1, -1))
    ex = [c[0] + 2 * c[3] * x + c[6] * y + c[7] * z, c[1] + 2 * c[4] * y + c[6] * x + c[8] * z,
          c[2] + 2 * c[5] * z + c[7] * x + c[8] * y]
    for a in range(3 if nz > 1 else 2):
        assert np.abs(grad[a][sl] - ex[a][sl]).max() < 1e-13
    lap_ex = 2 * (c[3] + c[4] + (c[5] if nz > 1 else 0))
    assert np.abs(lap[sl] - lap_ex).max() < 1e-12
    o.close()


def test_stencils_second_order_on_sine(oracle_mod):
    errs = []
    for n in (16, 32):
        P = wl.base_params(n, n, 1, phase_change=False, latent_heat=False)
        y, x = np.meshgrid(np.arange(n) + .5, np.arange(n) + .5, indexing="ij")
        k = 2 * np.pi / n
        phi = (np.sin(k * x) * np.cos(2 * k * y))[None]
        o = oracle_mod.Oracle(P)
        o.init(phi)
        grad, lap, _, _ = o.read_aux()
        e1 = np.abs(grad[0] - (k * np.cos(k * x) * np.cos(2 * k * y))[None]).max() / k
        e2 = np.abs(lap + 5 * k * k * phi).max() / (5 * k * k)
        errs.append((e1, e2))
        o.close()
    assert 3.5 < errs[0][0] / errs[1][0] < 4.5 and 3.5 < errs[0][1] / errs[1][1] < 4.5


# ---------------------------------------------------------------- P14 identities of the sources
@pytest.mark.parametrize("dims", [(8, 8, 1), (6, 6, 6)])
def test_source_moment_identities(oracle_mod, dims):
    """At init theta_bar = eq - dt/2 S, so post - bar = dt S exactly (Eq.25).  Then:
    sum_i S^f = c_s^2 u.grad rho + rho c_s^2 m''' Drho ; sum_i c_i S^f = c_s^2 F_tot ; sum eq_f = p ;
    sum c_i eq_f = rho c_s^2 u ; sum_i S^g = Pdot ; sum_i S^s = -(L/Cp) D ; the init moments return the inputs."""
    from test_oracle_bruteforce import _random_state
    P = wl.base_params(*dims, grav=[2e-4, -1e-4, 0.0], theta_I=0.02)
    phi, T, u, p = _random_state(P, 5)
    o = oracle_mod.Oracle(P)
    o.init(phi, T, u, p)
    grad, lap, pdot, _ = o.read_aux()
    e, w, e2 = oracle_mod.lattice(P["lat_f"])
    cs2 = e2
    bar = o.read_pops(0, oracle_mod.POPS_STREAMED)
    post = o.read_pops(0, oracle_mod.POPS_POSTCOLLISION)
    S = post - bar  # dt = 1
    feq = bar + 0.5 * S
    rho = phi * P["rho_g"] + (1 - phi) * P["rho_l"]
    grho = (P["rho_g"] - P["rho_l"]) * grad
    drho = 1 / P["rho_g"] - 1 / P["rho_l"]
    mdot = P["rho_g"] * pdot
    K, H = 1.5 * P["W"] * P["sigma"], 12 * P["sigma"] / P["W"]
    mu = 4 * H * phi * (phi - 1) * (phi - 0.5) - K * lap
    F = mu * grad + (rho - P["rho_l"]) * np.array(P["grav"]).reshape(3, 1, 1, 1)
    assert np.abs(S.sum(0) - (cs2 * (u * grho).sum(0) + rho * cs2 * mdot * drho)).max() < 1e-15
    for a in range(3):
        m1 = np.tensordot(e[:, a].astype(float), S, axes=(0, 0))
        assert np.abs(m1 - cs2 * F[a]).max() < 1e-15
        assert np.abs(np.tensordot(e[:, a].astype(float), feq, axes=(0, 0)) - rho * cs2 * u[a]).max() < 1e-15
    assert np.abs(feq.sum(0) - p).max() < 1e-15
    Sg = o.read_pops(1, oracle_mod.POPS_POSTCOLLISION) - o.read_pops(1, oracle_mod.POPS_STREAMED)
    assert np.abs(Sg.sum(0) - pdot).max() < 1e-15
    Ss = o.read_pops(2, oracle_mod.POPS_POSTCOLLISION) - o.read_pops(2, oracle_mod.POPS_STREAMED)
    D = (u * grad).sum(0) + phi * mdot * drho
    assert np.abs(Ss.sum(0) + (P["L_latent"] / P["Cp"]) * D).max() < 1e-14
    # Eq.(18) against a hand evaluation
    alpha = phi * P["alpha_g"] + (1 - phi) * P["alpha_l"]
    theta = P["Cp"] * (T - P["T_sat"]) / P["L_latent"]
    assert np.abs(pdot + 4 * alpha / (P["A"] * P["W"] ** 2) * (P["theta_I"] - theta) * phi * (1 - phi)).max() < 1e-15
    o.close()


# ---------------------------------------------------------------- P1 mass conservation, P3 CAC forms
def test_mass_conservation_periodic_and_walls(oracle_mod):
    """sum(phi) conserved to round-off when Pdot = 0, periodic box and zero-flux walls."""
    P, I = wl.config1_droplet(n=32, radius=8.0)
    o = oracle_mod.Oracle(P); o.init(I["phi"], I["T"])
    m0 = I["phi"].sum()
    o.step(300)
    assert abs(o.read_macro()[0].sum() - m0) / m0 < 1e-13
    o.close()
    P, I = wl.config3_film2d(nx=32, ny=48, h0=12.0, amp=2.0, phase_change=False, latent_heat=False)
    o = oracle_mod.Oracle(P); o.init(I["phi"], I["T"])
    m0 = I["phi"].sum()
    o.step(300)
    assert abs(o.read_macro()[0].sum() - m0) / m0 < 1e-13
    o.close()


def test_cac_source_form_equals_modified_equilibrium_form(oracle_mod):
    """P3, App. C.2: Eq.(29)-(30) and Eq.(31) give the same populations."""
    P, I = wl.config1_droplet(n=24, radius=6.0)
    P["phase_change"] = True
    I["T"] = I["T"] + 0.3
    a = oracle_mod.Oracle(P); a.init(I["phi"], I["T"])
    b = oracle_mod.Oracle(P); b.init(I["phi"], I["T"]); b.set_cac_form(oracle_mod.CAC_SOURCE)
    a.step(20); b.step(20)
    assert np.abs(a.read_pops(1) - b.read_pops(1)).max() < 1e-14
    assert np.abs(a.read_macro()[0] - b.read_macro()[0]).max() < 1e-14
    a.close(); b.close()


# ---------------------------------------------------------------- P17 symmetries
def test_3d_z_invariance_and_axis_permutation(oracle_mod):
    P, I = wl.config5_droplets(n=12, nspheres=3, rmin=2.0, rmax=4.0, seed=2)
    phi2d = I["phi"][0:1]
    T2d = I["T"][0:1]
    phi = np.repeat(phi2d, 12, axis=0); T = np.repeat(T2d, 12, axis=0)
    o = oracle_mod.Oracle(P); o.init(phi, T); o.step(15)
    ph, u, p, Tt = o.read_macro()
    assert np.abs(ph - ph[0:1]).max() < 1e-13 and np.abs(Tt - Tt[0:1]).max() < 1e-13
    assert np.abs(u[2]).max() < 1e-13
    o.close()
    # transposing the input x <-> z transposes the output
    o1 = oracle_mod.Oracle(P); o1.init(I["phi"], I["T"]); o1.step(15)
    o2 = oracle_mod.Oracle(P); o2.init(I["phi"].transpose(2, 1, 0).copy(), I["T"].transpose(2, 1, 0).copy()); o2.step(15)
    a, b = o1.read_macro(), o2.read_macro()
    assert np.abs(a[0] - b[0].transpose(2, 1, 0)).max() < 1e-12
    assert np.abs(a[3] - b[3].transpose(2, 1, 0)).max() < 1e-12
    assert np.abs(a[1][0] - b[1][2].transpose(2, 1, 0)).max() < 1e-12
    o1.close(); o2.close()
