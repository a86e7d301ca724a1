"""Seeded synthetic workloads: parameter dictionaries and initial fields of the five BASELINE.json configs.

This module is the ONE piece shared by the CUDA path, the CPU oracle and the tests.  It holds input
recipes only (grid shapes, boundary kinds, physical parameters, initial phi / T fields) and none of the
method's arithmetic: no lattice tables, no equilibria, no stencils.  All random numbers come from
``numpy.random.Generator(PCG64(seed))`` and are handed to both implementations as plain arrays.

Conventions: node (i, j, k) sits at ((i+1/2), (j+1/2), (k+1/2)) dx; dx = dt = 1;
arrays are x-fastest, shape (nz, ny, nx); phi = 1 is gas/vapour, phi = 0 liquid.
The initial interface profile is the paper's kernel function Eq.(7); the film-boiling
perturbation follows Eq.(42); parameter choices not fixed by BASELINE.json follow
SURVEY.md S11 and are recorded in every dictionary.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.special import erf

PER = "periodic"

# xi e^{xi^2} erf(xi) = St / sqrt(pi) for St = 0.1 (one-phase Stefan problem, config 2)
XI_STEFAN_ST01 = 0.220016


def base_params(nx, ny, nz=1, **over):
    """Defaults of SURVEY.md S11: rho_l/rho_g = 10, nu = 0.1 (tau_f = 0.8), M = 0.02, sigma = 1e-3, W = 4."""
    three_d = nz > 1
    P = dict(
        nx=int(nx), ny=int(ny), nz=int(nz),
        lat_f="D3Q19" if three_d else "D2Q9",
        lat_g="D3Q7" if three_d else "D2Q9",
        lat_s="D3Q7" if three_d else "D2Q5",
        bc_f=[[PER, PER], [PER, PER], [PER, PER]],
        bc_g=[[PER, PER], [PER, PER], [PER, PER]],
        bc_s=[[PER, PER], [PER, PER], [PER, PER]],
        bc_phi=[[0.0, 0.0], [0.0, 0.0], [0.0, 0.0]],
        bc_T=[[0.0, 0.0], [0.0, 0.0], [0.0, 0.0]],
        bc_p=[[0.0, 0.0], [0.0, 0.0], [0.0, 0.0]],
        dx=1.0, dt=1.0,
        rho_l=10.0, rho_g=1.0, nu_l=0.1, nu_g=0.1,
        sigma=1e-3, W=4.0, M=0.02,
        grav=[0.0, 0.0, 0.0],
        force=[0.0, 0.0, 0.0],
        alpha_l=0.02, alpha_g=0.05,
        L_latent=1.0, Cp=0.1, T_sat=0.0, theta_I=0.0,
        A=10.0 / 48.0, eps_n=1e-5,
        phase_change=True, latent_heat=True, prescribed_u=False,
    )
    P.update(over)
    return P


def _coords(P):
    nz, ny, nx = P["nz"], P["ny"], P["nx"]
    x = (np.arange(nx) + 0.5)[None, None, :]
    y = (np.arange(ny) + 0.5)[None, :, None]
    z = (np.arange(nz) + 0.5)[:, None, None]
    return x, y, z


def _noise(rng, shape, amp):
    return amp * rng.uniform(-1.0, 1.0, size=shape)


def config1_droplet(n=64, radius=16.0, seed=1, noise=1e-6, **over):
    """Config 1: 2D static liquid droplet in gas, n x n periodic, heat source off (BASELINE.json configs[0])."""
    P = base_params(n, n, 1, phase_change=False, latent_heat=False, **over)
    rng = np.random.Generator(np.random.PCG64(seed))
    x, y, _ = _coords(P)
    r = np.sqrt((x - n / 2.0) ** 2 + (y - n / 2.0) ** 2)
    phi = 0.5 * (1.0 - np.tanh(2.0 * (radius - r) / P["W"])) + _noise(rng, (1, n, n), noise)
    T = np.full((1, n, n), P["T_sat"])
    return P, dict(phi=phi, T=T, u=None, p=None, seed=seed, name="config1_droplet_%dx%d" % (n, n))


def config2_stefan(nx=512, ny=4, x_i0=32.0, open_right=True, **over):
    """Config 2: evaporating 1D Stefan strip, hot wall at x = 0, vapour for x < x_i0 (BASELINE.json configs[1]).

    The temperature starts on the one-phase similarity profile at the time t0 at which the analytic interface
    sits at x_i0, so the analytic position afterwards is 2 xi sqrt(alpha_g (t + t0))."""
    P = base_params(nx, ny, 1, **over)
    P["bc_f"][0] = ["wall", "open" if open_right else "wall"]
    P["bc_g"][0] = ["dirichlet", "dirichlet"]
    P["bc_s"][0] = ["dirichlet", "dirichlet"]
    P["bc_phi"][0] = [1.0, 0.0]
    T_w = P["T_sat"] + 1.0
    P["bc_T"][0] = [T_w, P["T_sat"]]
    P["bc_p"][0] = [0.0, 0.0]
    x, _, _ = _coords(P)
    xi = XI_STEFAN_ST01
    t0 = (x_i0 / (2.0 * xi)) ** 2 / P["alpha_g"]
    phi = 0.5 * (1.0 - np.tanh(2.0 * (x - x_i0) / P["W"])) + np.zeros((1, ny, 1))
    prof = P["T_sat"] + (T_w - P["T_sat"]) * (1.0 - erf(x / (2.0 * math.sqrt(P["alpha_g"] * t0))) / erf(xi))
    T = np.where(x < x_i0, prof, P["T_sat"]) + np.zeros((1, ny, 1))
    return P, dict(phi=phi, T=T, u=None, p=None, seed=None, t0=t0, xi=xi, name="config2_stefan_%dx%d" % (nx, ny))


def _film_bcs(P, axis):
    P["bc_f"][axis] = ["wall", "wall"]
    P["bc_g"][axis] = ["zeroflux", "zeroflux"]
    P["bc_s"][axis] = ["dirichlet", "dirichlet"]
    P["bc_T"][axis] = [P["T_sat"] + 1.0, P["T_sat"]]


def config3_film2d(nx=512, ny=1024, h0=64.0, amp=4.0, seed=3, noise=1e-6, modes=0, **over):
    """Config 3: 2D film boiling, x periodic, no-slip walls bottom/top, heated bottom wall (configs[2]).

    modes = 0: single-mode interface Eq.(42), one period across the box.  modes = m > 0: the multi-mode
    interface of the paper's 4096 x 3072 run, Eq.(44): h = h0 + amp sum_i sin(2 pi x / lambda_i) with m
    wavelengths drawn uniformly from [0.5, 1.5 sqrt(3)] lambda_c, lambda_c = 2 pi sqrt(sigma / ((rho_l - rho_g) g))
    (PAPER.md:526)."""
    P = base_params(nx, ny, 1, grav=[0.0, -1e-5, 0.0], **over)
    _film_bcs(P, 1)
    rng = np.random.Generator(np.random.PCG64(seed))
    x, y, _ = _coords(P)
    if modes > 0:
        lam_c = 2.0 * np.pi * math.sqrt(P["sigma"] / ((P["rho_l"] - P["rho_g"]) * abs(P["grav"][1])))
        lam = rng.uniform(0.5 * lam_c, 1.5 * math.sqrt(3.0) * lam_c, size=modes)
        h = h0 + amp * sum(np.sin(2.0 * np.pi * x / l) for l in lam)
    else:
        h = h0 + amp * np.sin(2.0 * np.pi * x / nx)
    phi = 0.5 * (1.0 - np.tanh(2.0 * (y - h) / P["W"])) + _noise(rng, (1, ny, nx), noise)
    T = P["T_sat"] + np.maximum(0.0, 1.0 - y / h)
    return P, dict(phi=phi, T=T, u=None, p=None, seed=seed, name="config3_film2d_%dx%d" % (nx, ny))


def paper_film_boiling(nx=1024, ny=1024, lam=0.64, seed=None, modes=0, y1=0.015, theta_w=0.025, **over):
    """The paper's own film-boiling set-up (Section 5), in ITS physical units: Table 2 parameters, domain
    [0, 1.28]^2 on 1024^2 nodes (dx = 1.25e-3, dt = 7.5e-5), three D2Q9 lattices, interface y = y0 + y1 sin(2 pi x / lambda) with
    y0 = 0.03, y1 = 0.015, lambda = 0.64 (Eq.42), bottom wall at theta_w = 0.025, top wall at saturation with
    phi = 1, x periodic.  With L/Cp = 1 and T_sat = 0 the temperature IS theta.  Not stated in the paper and chosen
    here: the initial temperature (conduction profile across the film, as in config 3) and the phase-field condition on the
    bottom wall (zero flux).  A smaller grid keeps dx, dt and the physical lengths (a window of the same problem).

    modes = 16 with nx, ny = 4096, 3072 is the paper's large run (Eq.44): y = y0 + y1 sum_i sin(2 pi x / lambda_i),
    lambda_i uniform in [0.5, 1.5 sqrt(3)] lambda_c (seeded), at theta_w = 0.025 or 0.1 (Ja = 0.025 / 0.1).  The paper does not restate
    y1 for that run; with sixteen modes y1 = 0.015 would put the interface below the wall, so pass a smaller y1 (the film is kept
    thicker than 2 W everywhere)."""
    dx, dt = 1.25e-3, 7.5e-5
    P = base_params(nx, ny, 1, lat_s="D2Q9", dx=dx, dt=dt, rho_l=1.658, rho_g=1.0, nu_l=3e-3, nu_g=5e-4,
                    alpha_l=2.5e-4, alpha_g=2.5e-3, sigma=5e-3, M=1.7e-3, W=5e-3, grav=[0.0, -4.0, 0.0],
                    L_latent=1.0, Cp=1.0, T_sat=0.0, theta_I=0.0, eps_n=1e-5 / dx, **over)
    P["bc_f"][1] = ["wall", "wall"]
    P["bc_g"][1] = ["zeroflux", "dirichlet"]
    P["bc_phi"][1] = [0.0, 1.0]
    P["bc_s"][1] = ["dirichlet", "dirichlet"]
    P["bc_T"][1] = [theta_w, 0.0]
    x = (np.arange(nx) + 0.5).reshape(1, 1, nx) * dx
    y = (np.arange(ny) + 0.5).reshape(1, ny, 1) * dx
    lam_s = math.sqrt(P["sigma"] / ((P["rho_l"] - P["rho_g"]) * 4.0))      # Eq.(43): 4.358e-2
    lam_c = 2.0 * math.pi * lam_s
    if modes > 0:
        rng = np.random.Generator(np.random.PCG64(44 if seed is None else seed))
        lams = rng.uniform(0.5 * lam_c, 1.5 * math.sqrt(3.0) * lam_c, size=modes)
        h = np.maximum(0.03 + y1 * sum(np.sin(2.0 * np.pi * x / l) for l in lams), 2.0 * P["W"])
    else:
        h = 0.03 + y1 * np.sin(2.0 * np.pi * x / lam)
    phi = 0.5 * (1.0 - np.tanh(2.0 * (y - h) / P["W"]))
    T = theta_w * np.maximum(0.0, 1.0 - y / h)
    return P, dict(phi=phi, T=T, u=None, p=None, seed=seed, t_s=math.sqrt(lam_s / 4.0), lam_c=lam_c,
                   name="paper_film_boiling_%dx%d" % (nx, ny))


def paper_film_boiling_3d(nx=256, ny=256, nz=384, y1=0.015, theta_w=0.025, **over):
    """The paper's film-boiling set-up carried to 3D (its 3D coupling terms were "planned"): Table 2 parameters
    in physical units (dx = 1.25e-3, dt = 7.5e-5), D3Q19 + D3Q7 + D3Q7, heated plate at z = 0, top wall at saturation with phi = 1,
    x and y periodic, film z = y0 + y1/2 [cos(2 pi x / Lx) + cos(2 pi y / Ly)] with y0 = 0.03: one crest per box.  The box must be
    wider than lambda_c = 0.2738 for the crest to grow (Eq.43): 256 nodes = 0.32."""
    dx, dt = 1.25e-3, 7.5e-5
    P = base_params(nx, ny, nz, dx=dx, dt=dt, rho_l=1.658, rho_g=1.0, nu_l=3e-3, nu_g=5e-4, alpha_l=2.5e-4, alpha_g=2.5e-3,
                    sigma=5e-3, M=1.7e-3, W=5e-3, grav=[0.0, 0.0, -4.0], L_latent=1.0, Cp=1.0, T_sat=0.0, theta_I=0.0,
                    eps_n=1e-5 / dx, **over)
    P["bc_f"][2] = ["wall", "wall"]
    P["bc_g"][2] = ["zeroflux", "dirichlet"]
    P["bc_phi"][2] = [0.0, 1.0]
    P["bc_s"][2] = ["dirichlet", "dirichlet"]
    P["bc_T"][2] = [theta_w, 0.0]
    x = (np.arange(nx) + 0.5).reshape(1, 1, nx) * dx
    y = (np.arange(ny) + 0.5).reshape(1, ny, 1) * dx
    z = (np.arange(nz) + 0.5).reshape(nz, 1, 1) * dx
    h = 0.03 + 0.5 * y1 * (np.cos(2.0 * np.pi * x / (nx * dx)) + np.cos(2.0 * np.pi * y / (ny * dx)))
    phi = 0.5 * (1.0 - np.tanh(2.0 * (z - h) / P["W"]))
    T = theta_w * np.maximum(0.0, 1.0 - z / h)
    lam_s = math.sqrt(P["sigma"] / ((P["rho_l"] - P["rho_g"]) * 4.0))
    return P, dict(phi=phi, T=T, u=None, p=None, seed=None, t_s=math.sqrt(lam_s / 4.0), lam_c=2.0 * math.pi * lam_s,
                   name="paper_film_boiling_3d_%dx%dx%d" % (nx, ny, nz))


def config4_film3d(nx=256, ny=256, nz=512, h0=32.0, amp=3.0, seed=4, zrange=None, **over):
    """Config 4: 3D film boiling, x,y periodic, walls in z, heated bottom plate (configs[3]).

    h(x,y) = h0 + amp/2 [cos(2 pi x/nx) + cos(2 pi y/ny)] + sum_k a_k sin(2 pi (m_k x/nx + n_k y/ny) + psi_k).
    zrange = (z0, z1): return the fields of layers z0..z1-1 only (one slab of a decomposed run); P is still global."""
    P = base_params(nx, ny, nz, grav=[0.0, 0.0, -1e-5], **over)
    _film_bcs(P, 2)
    rng = np.random.Generator(np.random.PCG64(seed))
    a = rng.uniform(0.0, 0.3, size=8)
    m = rng.integers(1, 5, size=8)
    n = rng.integers(1, 5, size=8)
    psi = rng.uniform(0.0, 2.0 * np.pi, size=8)
    x, y, z = _coords(P)
    h = h0 + 0.5 * amp * (np.cos(2.0 * np.pi * x / nx) + np.cos(2.0 * np.pi * y / ny))
    for k in range(8):
        h = h + a[k] * np.sin(2.0 * np.pi * (m[k] * x / nx + n[k] * y / ny) + psi[k])
    if zrange is not None:
        z = z[zrange[0]:zrange[1]]
    nzl = z.shape[0]
    phi = np.empty((nzl, ny, nx))
    T = np.empty((nzl, ny, nx))
    for k0 in range(0, nzl, 32):  # chunks keep the temporaries small at 256x256x512
        zz = z[k0:k0 + 32]
        phi[k0:k0 + 32] = 0.5 * (1.0 - np.tanh(2.0 * (zz - h) / P["W"]))
        T[k0:k0 + 32] = P["T_sat"] + np.maximum(0.0, 1.0 - zz / h)
    return P, dict(phi=phi, T=T, u=None, p=None, seed=seed, name="config4_film3d_%dx%dx%d" % (nx, ny, nz))


def config5_droplets(n=128, nspheres=64, rmin=8.0, rmax=24.0, seed=5, **over):
    """Config 5: cubic periodic box with a seeded random field of liquid droplets, T noise (configs[4])."""
    P = base_params(n, n, n, **over)
    rng = np.random.Generator(np.random.PCG64(seed))
    cen = rng.uniform(0.0, n, size=(nspheres, 3))
    rad = rng.uniform(rmin, rmax, size=nspheres)
    x, y, z = _coords(P)
    phi = np.empty((n, n, n))
    for k0 in range(0, n, 8):
        zz = z[k0:k0 + 8]
        d = np.full((zz.shape[0], n, n), -np.inf)
        for c, R in zip(cen, rad):
            ddx = np.abs(x - c[0]); ddx = np.minimum(ddx, n - ddx)
            ddy = np.abs(y - c[1]); ddy = np.minimum(ddy, n - ddy)
            ddz = np.abs(zz - c[2]); ddz = np.minimum(ddz, n - ddz)
            d = np.maximum(d, R - np.sqrt(ddx * ddx + ddy * ddy + ddz * ddz))
        phi[k0:k0 + 8] = 0.5 * (1.0 - np.tanh(2.0 * d / P["W"]))
    T = P["T_sat"] + rng.uniform(-0.5, 0.5, size=(n, n, n))
    return P, dict(phi=phi, T=T, u=None, p=None, seed=seed, name="config5_droplets_%d^3" % n)


def bytes_per_lu(P, itemsize=8, macros=False):
    """Algorithmic HBM bytes per lattice update of the two-kernel step.

    K_phi: Q_g reads, 1 write (the dt/2 Pdot term of Eq.32 rides in the stored rest population of g).  K_main: Q_f + Q_g + Q_s + 3 reads (phi^{n+1}, phi^n, Pdot),
    Q_f + Q_g + Q_s + 1 writes (+5 or +4 when u, p, T are written).  The three phi values (one written, two read) are
    doubles in both precisions (include/lbm.h "Precisions")."""
    q = {"D2Q5": 5, "D2Q9": 9, "D3Q7": 7, "D3Q19": 19, "D3Q15": 15}
    Q = q[P["lat_f"]] + q[P["lat_g"]] + q[P["lat_s"]]
    vals = (q[P["lat_g"]] + 1) + (Q + 3) + (Q + 1)
    if macros:
        vals += (3 if P["nz"] > 1 else 2) + 2
    return vals * itemsize + 3 * (8 - itemsize)
