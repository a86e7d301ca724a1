"""Run the BASELINE.json configurations at their FULL step counts on the GPU and report physical observables.

    python -m paper_2003_06342_b200.run_configs [--configs 1,2,3,3_window,4,stefan_paper,paper,paper_full,paper_3d,paper_large,paper_large_ja01] [--set M=0.1] [--precision 64] [--samples 10]

One JSON line per configuration: the observables the paper discusses for that test (PAPER.md:446 Laplace law, PAPER.md:473
Stefan interface position, PAPER.md:535 bubbles growing and rising from the heated wall) sampled along the run, plus
sum(phi) and the finiteness of every field.  Everything is computed by the library's kernels; this module only samples
`lbm_read_macro` and reduces the host arrays (argument marshalling and post-processing, no arithmetic of the method).
The parity statements of the repository are made against the CPU oracle at the horizons of DESIGN.md "Parity horizon";
beyond them a film-boiling run is a physical instability and is compared on observables such as these.
"""
from __future__ import annotations

import argparse
import json
import math
import time

import numpy as np

from . import binding, workloads as wl


def interface_x(phi_row):
    """Position (node units, node i at i + 1/2) where phi crosses 1/2 along a row that starts in vapour (phi = 1)."""
    below = np.nonzero(phi_row < 0.5)[0]
    if len(below) == 0 or below[0] == 0:
        return float("nan")
    i = int(below[0])
    a, b = float(phi_row[i - 1]), float(phi_row[i])
    return (i - 1 + 0.5) + (a - 0.5) / (a - b)


def film_thickness(phi):
    """Per column: number of vapour nodes (phi > 1/2) between the heated wall and the first liquid node; wall-normal axis first."""
    liquid = phi <= 0.5
    first = liquid.argmax(axis=0).astype(np.float64)
    first[~liquid.any(axis=0)] = phi.shape[0]
    return first


def detached_bubbles(phi):
    """(count, highest node, nodes) of the connected vapour regions that touch neither the heated wall nor the opposite wall."""
    from scipy import ndimage
    lab, n = ndimage.label(phi > 0.5)
    if n == 0:
        return 0, 0, 0
    attached = set(np.unique(lab[0])) | set(np.unique(lab[-1]))
    free = [k for k in range(1, n + 1) if k not in attached]
    if not free:
        return 0, 0, 0
    mask = np.isin(lab, free)
    top = int(np.nonzero(mask.reshape(mask.shape[0], -1).any(axis=1))[0].max()) + 1
    return len(free), top, int(mask.sum())


def run_config1(prec, samples):
    P, I = wl.config1_droplet()
    steps = 1000
    sim = binding.LBM(P, prec)
    dt = sim.dtype
    sim.init(I["phi"].astype(dt), I["T"].astype(dt))
    mass0 = float(I["phi"].astype(np.float64).sum())
    out = []
    every = max(1, steps // samples)
    for k in range(0, steps, every):
        sim.step(every)
        phi, u, p, T = sim.read_macro()
        inside = float(p[0, 28:36, 28:36].mean())                     # liquid drop (phi = 0) around the centre
        outside = float(np.concatenate([p[0, :4, :].ravel(), p[0, -4:, :].ravel()]).mean())
        out.append(dict(step=sim.step_count, laplace_ratio=(inside - outside) / (P["sigma"] / 16.0),
                        mass_drift=abs(float(phi.astype(np.float64).sum()) - mass0) / mass0,
                        umax=float(np.abs(u).max())))
    sim.destroy()
    return dict(config=1, name=I["name"], steps=steps, samples=out,
                note="Laplace law dp = sigma/R (PAPER.md:446): still ringing acoustically at 1000 steps, 0.93 when converged (DESIGN.md)")


def run_config2(prec, samples):
    P, I = wl.config2_stefan()
    steps = 20000
    sim = binding.LBM(P, prec)
    dt = sim.dtype
    sim.init(I["phi"].astype(dt), I["T"].astype(dt))
    out = []
    every = max(1, steps // samples)
    for k in range(0, steps, every):
        sim.step(every)
        phi, u, p, T = sim.read_macro()
        t = sim.step_count
        out.append(dict(step=t, x_interface=interface_x(phi[0, 0, :]),
                        x_analytic=2.0 * I["xi"] * math.sqrt(P["alpha_g"] * (t + I["t0"])),
                        y_spread=float(np.abs(phi[0] - phi[0, :1]).max())))
    sim.destroy()
    return dict(config=2, name=I["name"], steps=steps, samples=out,
                note="one-phase Stefan solution x_I = 2 xi sqrt(alpha_g (t + t0)), xi = 0.220016 (SURVEY.md S12); with the Navier-Stokes "
                     "lattice on and the OPEN face the interface runs 0.3 cell ahead at 20 000 steps (DESIGN.md)")


def run_stefan_paper(prec, samples):
    """The paper's Stefan validation (Fig.7): 512 x 32, D2Q9 for phi and T, flow at rest (equal densities, no
    surface tension), W = 3, M = 0.08, theta_w = -0.3, theta_inf = 0.3, t_f = 2e5 steps; interface position against
    x_I = 2 xi sqrt(alpha_l t) (Eq.41a) with the xi the paper prints for its six cases."""
    cases = [(0.14, 0.14, 0.0, 0.280680), (0.08, 0.08, 0.0, 0.280680), (0.03, 0.03, 0.0, 0.280680),
             (0.14, 0.014, 0.05, 0.349635), (0.125, 0.025, 0.05, 0.343882), (0.08, 0.04, 0.05, 0.331864)]
    nx, ny, steps = 512, 32, 200000
    out = []
    for alpha_l, alpha_g, theta_I, xi in cases:
        P = wl.base_params(nx, ny, 1, lat_s="D2Q9", rho_l=1.0, rho_g=1.0, sigma=0.0, W=3.0, M=0.08, Cp=1.0, L_latent=1.0,
                           alpha_l=alpha_l, alpha_g=alpha_g, theta_I=theta_I)
        P["bc_f"][0] = ["wall", "wall"]
        P["bc_g"][0] = ["dirichlet", "dirichlet"]
        P["bc_s"][0] = ["dirichlet", "dirichlet"]
        P["bc_phi"][0] = [0.0, 1.0]
        P["bc_T"][0] = [-0.3, 0.3]
        x = (np.arange(nx) + 0.5)[None, None, :]
        phi0 = 0.5 * (1.0 + np.tanh(2.0 * x / 3.0)) + np.zeros((1, ny, 1))
        sim = binding.LBM(P, prec)
        sim.init(phi0.astype(sim.dtype), np.full((1, ny, nx), 0.3, dtype=sim.dtype))
        rows = []
        every = steps // samples
        for k in range(samples):
            sim.step(every)
            phi = sim.read_macro()[0]
            row = phi[0, 0, :]
            j = int(np.nonzero((row[:-1] < 0.5) & (row[1:] >= 0.5))[0][0])          # liquid (phi = 0) grows from the cold wall
            x_i = (j + 0.5) + (0.5 - float(row[j])) / (float(row[j + 1]) - float(row[j]))
            t = sim.step_count
            rows.append(dict(step=t, x_interface=x_i, x_analytic=2.0 * xi * math.sqrt(alpha_l * t),
                             ratio=x_i / (2.0 * xi * math.sqrt(alpha_l * t))))
        sim.destroy()
        out.append(dict(alpha_l=alpha_l, alpha_g=alpha_g, theta_I=theta_I, xi=xi, samples=rows))
    return dict(config="stefan_paper", name="paper_stefan_512x32", steps=steps, cases=out,
                note="PAPER.md:498-500: xi = 0.280680 for theta_I = 0; 0.349635 / 0.343882 / 0.331864 for alpha_l/alpha_g = 10 / 5 / 2, theta_I = 0.05")


def _run_film(config, P, I, steps, prec, samples, normal_axis):
    sim = binding.LBM(P, prec)
    dt = sim.dtype
    sim.init(I["phi"].astype(dt), I["T"].astype(dt))
    out = []
    every = max(1, steps // samples)
    t_start = time.perf_counter()
    for k in range(0, steps, every):
        sim.step(every)
        phi, u, p, T = sim.read_macro()
        ph = phi if P["nz"] > 1 else phi[0]           # wall-normal axis first in both cases
        finite = bool(np.isfinite(phi).all() and np.isfinite(T).all() and np.isfinite(u).all())
        if not finite:
            out.append(dict(step=sim.step_count, finite=False))
            break
        h = film_thickness(ph)
        nb, btop, bnodes = detached_bubbles(ph)
        un = u[2] if P["nz"] > 1 else u[1]
        out.append(dict(step=sim.step_count, vapour_volume=float(ph.astype(np.float64).sum()),
                        h_mean=float(h.mean()), h_max=float(h.max()), h_min=float(h.min()),
                        bubbles=nb, bubble_top=btop, bubble_nodes=bnodes,
                        u_normal_max=float(un.max()), u_normal_min=float(un.min()),
                        T_min=float(T.min()), T_max=float(T.max()), phi_min=float(phi.min()), phi_max=float(phi.max()),
                        finite=True))
    wall = time.perf_counter() - t_start
    sim.destroy()
    return dict(config=config, name=I["name"], steps=steps, samples=out, wall_seconds_including_reads=wall,
                note="film boiling (PAPER.md:520-535): the vapour film thickens by evaporation at the heated wall, the crest of the "
                     "perturbation grows (Rayleigh-Taylor), bubbles rise: h_max (thickness of the attached film) and the vapour volume "
                     "increase, u_normal_max > 0; the run stops at the first non-finite sample")


def run_config3(prec, samples):
    P, I = wl.config3_film2d()
    return _run_film(3, P, I, 50000, prec, samples, 0)


def run_config3_window(prec, samples, **over):
    """Config 3 on a 128 x 256 window (film height 32) for 30 000 steps: small enough for the oracle to follow
    (tests/test_gpu_parity.py::test_config3_window_diverges_like_the_oracle); `--set key=value` varies one parameter."""
    P, I = wl.config3_film2d(nx=128, ny=256, h0=32.0, amp=4.0, **over)
    r = _run_film("3_window", P, I, 30000, prec, samples, 0)
    r["overrides"] = over
    return r


def run_config4(prec, samples):
    P, I = wl.config4_film3d()
    return _run_film(4, P, I, 5000, prec, samples, 0)


def run_paper_film(prec, samples, steps=200000, label="paper", **kw):
    """The paper's film-boiling run (Table 2, 1024^2); the paper ran 5.33e5 steps, a bubble cycle shows much earlier."""
    P, I = wl.paper_film_boiling(**kw)
    r = _run_film(label, P, I, steps, prec, samples, 0)
    for s in r["samples"]:
        s["t_star"] = s["step"] * P["dt"] / I["t_s"]          # dimensionless time of PAPER.md:535
        for k in ("h_mean", "h_max", "h_min", "bubble_top"):
            if k in s:
                s[k] *= P["dx"]                                # physical heights
        if "vapour_volume" in s:
            s["vapour_volume"] *= P["dx"] ** 2
    r["lambda_c"], r["t_s"] = I["lam_c"], I["t_s"]
    r["note"] = ("paper's set-up: lambda = 0.64 > lambda_c = 0.2738, bubbles grow on the two crests ('nodes'), detach and rise, then on the "
                 "anti-nodes (PAPER.md:535): `bubbles` counts the detached vapour regions, `bubble_top` their highest point in the domain "
                 "[0, 1.28]; h_* is the thickness of the film still attached to the heated wall")
    return r


def run_paper_large(prec, samples, theta_w=0.025):
    """The paper's 8-GPU run: 4096 x 3072, sixteen modes (Eq.44), 5.33e5 steps, on one GPU."""
    r = run_paper_film(prec, samples, steps=533000, label="paper_large_Ja%g" % theta_w, nx=4096, ny=3072, modes=16, y1=0.004,
                       theta_w=theta_w)
    r["mlups_including_reads"] = 4096.0 * 3072.0 * 533000 / r["wall_seconds_including_reads"] / 1e6
    r["note"] = ("PAPER.md:563: 80 minutes on 8 GPUs (713 MLUPS as printed) for these 5.33e5 steps; Ja = 0.025 releases discrete bubbles, "
                 "Ja = 0.1 grows long vapour jets under the bubbles (h_max: the film still attached to the wall reaches far up)")
    return r


def run_paper_3d(prec, samples, steps=60000):
    """The paper's film boiling carried to 3D (workloads.paper_film_boiling_3d): the coupling terms the paper left for later."""
    P, I = wl.paper_film_boiling_3d()
    r = _run_film("paper_3d", P, I, steps, prec, samples, 0)
    for s in r["samples"]:
        s["t_star"] = s["step"] * P["dt"] / I["t_s"]
        for k in ("h_mean", "h_max", "h_min", "bubble_top"):
            if k in s:
                s[k] *= P["dx"]
        if "vapour_volume" in s:
            s["vapour_volume"] *= P["dx"] ** 3
    r["note"] = "3D film boiling with the paper's Table 2 parameters: one crest per periodic box of 0.32 x 0.32, domain height 0.48"
    return r


RUNNERS = {1: run_config1, 2: run_config2, 3: run_config3, 4: run_config4, "paper": run_paper_film,
           "stefan_paper": run_stefan_paper, "paper_full": lambda prec, samples: run_paper_film(prec, samples, steps=533000, label="paper_full"), "paper_3d": run_paper_3d, "paper_large": run_paper_large, "paper_large_ja01": lambda prec, samples: run_paper_large(prec, samples, theta_w=0.1)}


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--configs", default="1,2,3,4")
    ap.add_argument("--precision", type=int, default=64, choices=(32, 64))
    ap.add_argument("--samples", type=int, default=10)
    ap.add_argument("--set", action="append", default=[], metavar="KEY=VALUE", help="3_window only: override a physical parameter")
    args = ap.parse_args(argv)
    binding.load_library()
    for c in args.configs.split(","):
        if c == "3_window":
            over = {kv.split("=")[0]: float(kv.split("=")[1]) for kv in args.set}
            print(json.dumps(run_config3_window(args.precision, args.samples, **over)), flush=True)
            continue
        key = c if (c.startswith("paper") or c.startswith("stefan")) else int(c)
        print(json.dumps(RUNNERS[key](args.precision, args.samples)), flush=True)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
