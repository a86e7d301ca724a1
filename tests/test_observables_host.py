"""Host logic of the observables helpers (tests/observables.py) and of the paper's film-boiling recipe: no GPU, no
arithmetic of the method -- the reductions that turn fields into the observables of PAPER.md:535."""
import math

import numpy as np

import observables as rc
from paper_2003_06342_b200 import workloads as wl


def test_interface_position_by_linear_interpolation():
    x = np.arange(64) + 0.5
    phi = 0.5 * (1.0 - np.tanh(2.0 * (x - 20.3) / 4.0))
    assert abs(rc.interface_x(phi) - 20.3) < 0.02
    assert math.isnan(rc.interface_x(np.zeros(8)))          # no vapour at the wall


def test_film_thickness_and_detached_bubbles():
    phi = np.zeros((40, 30))
    phi[:5, :] = 1.0                     # film of 5 nodes on the heated wall
    phi[:9, 10:12] = 1.0                 # a crest of 9 nodes
    phi[20:24, 5:9] = 1.0                # a free bubble
    phi[30:33, 20:22] = 1.0              # another one, higher
    phi[-2:, :] = 1.0                    # gas layer under the opposite wall (the paper's top boundary)
    h = rc.film_thickness(phi)
    assert h.min() == 5 and h.max() == 9 and h[0] == 5 and h[10] == 9
    n, top, nodes = rc.detached_bubbles(phi)
    assert (n, top, nodes) == (2, 33, 16 + 6)
    assert rc.detached_bubbles(np.zeros((8, 8))) == (0, 0, 0)
    # 3D: wall-normal axis first
    phi3 = np.zeros((20, 6, 7)); phi3[:3] = 1.0; phi3[10:12, 2:4, 2:4] = 1.0
    assert rc.film_thickness(phi3).shape == (6, 7) and rc.detached_bubbles(phi3)[0] == 1


def test_paper_film_boiling_recipe():
    """Table 2 and Eq.(42)-(44) of the paper."""
    P, I = wl.paper_film_boiling(nx=512, ny=128)           # one wavelength, lambda = 0.64 = 512 dx
    assert (P["dx"], P["dt"]) == (1.25e-3, 7.5e-5) and P["lat_s"] == "D2Q9"
    assert abs(I["lam_c"] - 0.2738) < 1e-4 and abs(I["t_s"] - 0.1044) < 1e-4          # values printed at PAPER.md:531, 535
    c = P["dx"] / P["dt"]
    cs2 = c * c / 3.0
    for nu in (P["nu_l"], P["nu_g"], P["M"], P["alpha_l"], P["alpha_g"]):
        assert nu / (cs2 * P["dt"]) > 0.03                                              # every relaxation time is resolvable
    phi = I["phi"][0]
    h = (phi > 0.5).sum(axis=0) * P["dx"]
    assert abs(h.mean() - 0.03) < 2e-3 and abs(h.max() - 0.045) < 2e-3                  # y0 = 0.03, y1 = 0.015
    assert I["T"].max() <= 0.025 and I["T"].min() == 0.0
    assert P["bc_T"][1] == [0.025, 0.0] and P["bc_g"][1] == ["zeroflux", "dirichlet"] and P["bc_phi"][1][1] == 1.0
    # sixteen modes: seeded, the film never thinner than 2 W
    P2, I2 = wl.paper_film_boiling(nx=1024, ny=64, modes=16, y1=0.004, theta_w=0.1)
    _, I3 = wl.paper_film_boiling(nx=1024, ny=64, modes=16, y1=0.004, theta_w=0.1)
    assert np.array_equal(I2["phi"], I3["phi"]) and I2["T"].max() <= 0.1
    assert ((I2["phi"][0] > 0.5).sum(axis=0) * P2["dx"]).min() >= 2 * P2["W"] - P2["dx"]


def test_paper_film_boiling_3d_recipe():
    P, I = wl.paper_film_boiling_3d(nx=32, ny=32, nz=48)
    assert (P["lat_f"], P["lat_g"], P["lat_s"]) == ("D3Q19", "D3Q7", "D3Q7") and P["grav"] == [0.0, 0.0, -4.0]
    assert I["phi"].shape == (48, 32, 32) and P["bc_phi"][2] == [0.0, 1.0] and P["bc_T"][2] == [0.025, 0.0]
    h = (I["phi"] > 0.5).sum(axis=0) * P["dx"]
    assert abs(h.max() - 0.045) < 2e-3 and abs(h.min() - 0.015) < 2e-3 and abs(h.mean() - 0.03) < 1e-3   # y0 +- y1, one crest per box
