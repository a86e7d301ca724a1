"""Pins of the model variants of SURVEY.md 8(f) #4 that the paper defines: the biased directional derivatives of
PAPER.md:318 inside the gradient Eq.(35b) (``grad_scheme``), and the stencil divergence of u phi as the alternative to the
product rule of reading S5 (``div_scheme``, reading S17; Eq.(33d), (34)).  Each test says which
plausible mistake it catches."""
import numpy as np
import pytest

from np_bruteforce import NPModel
from paper_2003_06342_b200 import workloads as wl
from test_oracle_bruteforce import _compare, _random_state


def _grad(oracle_mod, P, phi):
    o = oracle_mod.Oracle(P)
    o.init(phi)
    grad, lap, _, _ = o.read_aux()
    o.close()
    return grad, lap


@pytest.mark.parametrize("dims", [(12, 10, 1), (9, 8, 7)])
def test_biased1_gradient_is_the_central_gradient(oracle_mod, dims):
    """sum_i w_i e_i = 0, so the first-order biased difference [phi(x+e) - phi(x)]/dx of PAPER.md:318, assembled by Eq.(35b)
    over ALL directions, IS the central gradient: sum_i w_i e_i phi(x+e_i)/dx in both cases.  Catches: phi(x-e) taken for
    phi(x+e), a missing 1/dx or a factor 2, weights of another lattice, a sum that skips directions."""
    rng = np.random.Generator(np.random.PCG64(5))
    phi = rng.uniform(0, 1, dims[::-1])
    for lat_f in (("D3Q19", "D3Q15") if dims[2] > 1 else ("D2Q9",)):
        P = wl.base_params(*dims, dx=0.5, dt=0.5, phase_change=False, latent_heat=False, lat_f=lat_f)
        gc, lc = _grad(oracle_mod, P, phi)
        gb, lb = _grad(oracle_mod, dict(P, grad_scheme="biased1"), phi)
        assert np.abs(gb - gc).max() < 1e-13 and np.abs(gc).max() > 0.1
        assert np.array_equal(lb, lc)      # the Laplacian is Eq.(36) whatever the gradient scheme


@pytest.mark.parametrize("dims", [(12, 10, 1), (9, 8, 7)])
def test_biased2_gradient_exact_on_quadratics(oracle_mod, dims):
    """[-phi(x+2e) + 4 phi(x+e) - 3 phi(x)]/(2 dx) is exact for quadratics along e, so is the assembled
    gradient, two nodes away from the (zero-flux) faces.  Catches a wrong coefficient (-1, 4, -3), a wrong denominator
    and a second neighbour taken at x+e instead of x+2e."""
    P = wl.base_params(*dims, phase_change=False, latent_heat=False, grad_scheme="biased2")
    for a in range(3 if dims[2] > 1 else 2):
        P["bc_f"][a] = ["wall", "wall"]; P["bc_g"][a] = ["zeroflux", "zeroflux"]; P["bc_s"][a] = ["zeroflux", "zeroflux"]
    nz, ny, nx = dims[::-1]
    z, y, x = np.meshgrid(np.arange(nz) + .5, np.arange(ny) + .5, np.arange(nx) + .5, indexing="ij")
    c = [0.3, -0.2, 0.15, 0.01, -0.02, 0.005, 0.007, -0.004, 0.003]
    if nz == 1:
        z = 0 * z
    phi = c[0] * x + c[1] * y + c[2] * z + c[3] * x * x + c[4] * y * y + c[5] * z * z + c[6] * x * y + c[7] * x * z + c[8] * y * z
    grad, _ = _grad(oracle_mod, P, phi)
    sl = (slice(2, -2) if nz > 1 else slice(None), slice(2, -2), slice(2, -2))
    ex = [c[0] + 2 * c[3] * x + c[6] * y + c[7] * z, c[1] + 2 * c[4] * y + c[6] * x + c[8] * z,
          c[2] + 2 * c[5] * z + c[7] * x + c[8] * y]
    for a in range(3 if nz > 1 else 2):
        assert np.abs(grad[a][sl] - ex[a][sl]).max() < 1e-13


def test_biased2_gradient_closed_form_on_a_sine(oracle_mod):
    """For phi = sin(kx) the assembled second-order biased gradient is cos(kx) [4 sin(kh) - sin(2kh)]/(2h) (pairs e, -e:
    w e {4[phi(x+h) - phi(x-h)] - [phi(x+2h) - phi(x-2h)]}/(2h), and sum_i w_i e_ix^2 = e2), i.e. k cos(kx) (1 + k^2 h^2/3 + ...):
    second order with the OPPOSITE sign of the central error (1 - k^2 h^2/6).  Closed form to round-off; order from two grids."""
    errs = []
    for n in (16, 32):
        P = wl.base_params(n, 6, 1, phase_change=False, latent_heat=False, grad_scheme="biased2")
        x = (np.arange(n) + .5)[None, None, :] + np.zeros((1, 6, 1))
        k = 2 * np.pi / n
        grad, _ = _grad(oracle_mod, P, np.sin(k * x))
        closed = np.cos(k * x) * (4 * np.sin(k) - np.sin(2 * k)) / 2
        assert np.abs(grad[0] - closed).max() < 1e-14 and np.abs(grad[1]).max() < 1e-15
        errs.append(np.abs(grad[0] - k * np.cos(k * x)).max() / k)
    assert 3.6 < errs[0] / errs[1] < 4.2 and abs(errs[1] / ((2 * np.pi / 32) ** 2 / 3) - 1) < 0.05


def test_biased2_ghost_layers(oracle_mod):
    """The second neighbour beyond a face (reading S8-iv carried two deep): periodic wrap; zero-flux face phi(-2) = phi(1);
    Dirichlet face phi(-2) = 2v - phi(1).  Checked at the wall nodes against the NumPy model, which builds its ghost layers
    by flipping slabs (not by index arithmetic), and on a field whose exact gradient at the wall node is known: phi = v + s y
    through a Dirichlet face at y = 0 is continued linearly by 2v - mirror, so the biased gradient there is exactly s."""
    P = wl.base_params(10, 9, 1, phase_change=False, latent_heat=False, grad_scheme="biased2")
    P["bc_f"][1] = ["wall", "wall"]; P["bc_g"][1] = ["dirichlet", "zeroflux"]; P["bc_s"][1] = ["zeroflux", "zeroflux"]
    P["bc_phi"][1] = [0.25, 0.0]
    y = (np.arange(9) + .5)[None, :, None] + np.zeros((1, 1, 10))
    grad, _ = _grad(oracle_mod, P, 0.25 + 0.03 * y)
    assert np.abs(grad[1][0, :7] - 0.03).max() < 1e-14          # including the two layers next to the Dirichlet face
    assert abs(grad[1][0, 8, 0] - 0.03) > 1e-3                   # the zero-flux mirror bends the profile at the other face
    rng = np.random.Generator(np.random.PCG64(6))
    phi = rng.uniform(0, 1, (1, 9, 10))
    grad, _ = _grad(oracle_mod, P, phi)
    m = NPModel(P)
    g2, _ = m.derive(phi)
    assert np.abs(grad - g2).max() < 1e-13


def _div(oracle_mod, P, phi, u):
    o = oracle_mod.Oracle(P)
    o.init(phi, None, u, None)
    d = o.read_div()
    grad, _, _, _ = o.read_aux()
    o.close()
    return d, grad


@pytest.mark.parametrize("dims", [(12, 10, 1), (9, 8, 7)])
def test_stencil_divergence_of_a_uniform_velocity_is_u_dot_central_gradient(oracle_mod, dims):
    """div(u0 phi) by the stencil = u0 . grad(phi) by Eq.(35a,b): the two discretisations of reading S5 / S17 coincide when
    div u = 0 and u is uniform.  Catches a transposed e_i . u, a wrong 1/e2, a missing direction."""
    rng = np.random.Generator(np.random.PCG64(7))
    shape = dims[::-1]
    phi = rng.uniform(0, 1, shape)
    u = np.zeros((3,) + shape)
    u0 = [0.03, -0.02, 0.05 if dims[2] > 1 else 0.0]
    for a in range(3):
        u[a] = u0[a]
    for lat_f in (("D3Q19", "D3Q15") if dims[2] > 1 else ("D2Q9",)):
        P = wl.base_params(*dims, dx=0.5, dt=0.5, phase_change=False, prescribed_u=True, div_scheme="stencil", lat_f=lat_f)
        d, grad = _div(oracle_mod, P, phi, u)
        assert np.abs(d - sum(u0[a] * grad[a] for a in range(3))).max() < 1e-14


def test_stencil_divergence_exact_on_quadratic_flux_and_closed_form_on_sines(oracle_mod):
    """u linear, phi linear: u phi is quadratic and the central stencil exact (interior).  u = (sin kx, 0), phi = 1:
    div = cos(kx) sin(kh)/h to round-off.  Catches phi taken at the centre instead of the neighbour, u at the centre."""
    nx, ny = 14, 12
    P = wl.base_params(nx, ny, 1, phase_change=False, prescribed_u=True, div_scheme="stencil")
    for a in range(2):
        P["bc_f"][a] = ["wall", "wall"]; P["bc_g"][a] = ["zeroflux", "zeroflux"]; P["bc_s"][a] = ["zeroflux", "zeroflux"]
    y, x = np.meshgrid(np.arange(ny) + .5, np.arange(nx) + .5, indexing="ij")
    phi = (0.2 + 0.03 * x - 0.01 * y)[None]
    u = np.zeros((3, 1, ny, nx))
    u[0, 0] = 0.01 + 0.002 * x + 0.001 * y
    u[1, 0] = -0.02 + 0.003 * x - 0.004 * y
    d, _ = _div(oracle_mod, P, phi, u)
    exact = 0.002 * phi[0] + u[0, 0] * 0.03 - 0.004 * phi[0] + u[1, 0] * (-0.01)
    assert np.abs(d[0, 1:-1, 1:-1] - exact[1:-1, 1:-1]).max() < 1e-15
    n = 24
    P = wl.base_params(n, 6, 1, phase_change=False, prescribed_u=True, div_scheme="stencil")
    x = (np.arange(n) + .5)[None, None, :] + np.zeros((1, 6, 1))
    k = 2 * np.pi / n
    u = np.zeros((3, 1, 6, n)); u[0] = np.sin(k * x)
    d, _ = _div(oracle_mod, P, np.ones((1, 6, n)), u)
    assert np.abs(d - np.cos(k * x) * np.sin(k)).max() < 1e-15


def test_stencil_divergence_wall_and_open_ghost_velocity(oracle_mod):
    """Reading S17: beyond a no-slip wall the velocity is reflected ODD (zero on the wall, half a cell outside the first
    node), beyond an open face EVEN.  u_y = y (zero on the wall y = 0), phi = 1: d_y(u_y phi) = 1 at the wall node as well;
    an even reflection there would give 1/2.  At the open face on top the even reflection gives (u(n-1) - u(n-2))/2 = 1/2."""
    nx, ny = 6, 10
    P = wl.base_params(nx, ny, 1, phase_change=False, prescribed_u=True, div_scheme="stencil")
    P["bc_f"][1] = ["wall", "open"]; P["bc_g"][1] = ["zeroflux", "zeroflux"]; P["bc_s"][1] = ["zeroflux", "zeroflux"]
    y = (np.arange(ny) + .5)[None, :, None] + np.zeros((1, 1, nx))
    u = np.zeros((3, 1, ny, nx)); u[1] = y
    d, _ = _div(oracle_mod, P, np.ones((1, ny, nx)), u)
    assert np.abs(d[0, :-1] - 1.0).max() < 1e-15
    assert np.abs(d[0, -1] - 0.5).max() < 1e-15


def test_variants_against_the_numpy_model(oracle_mod):
    """Brute force: the full coupled step with each scheme against the independent NumPy transcription (np.pad-style ghost
    slabs, whole-array stencils) on tiny grids with every boundary kind, 2D and 3D."""
    for over in (dict(grad_scheme="biased1"), dict(grad_scheme="biased2"), dict(div_scheme="stencil"),
                 dict(grad_scheme="biased2", div_scheme="stencil")):
        P = wl.base_params(8, 8, 1, grav=[1e-4, -2e-4, 0.0], nu_l=0.05, nu_g=0.2, **over)
        _compare(oracle_mod, P, 10, 11)
        P = wl.base_params(8, 8, 1, grav=[0.0, -1e-4, 0.0], **over)
        P["bc_f"][1] = ["wall", "open"]; P["bc_g"][1] = ["zeroflux", "dirichlet"]; P["bc_s"][1] = ["dirichlet", "zeroflux"]
        P["bc_phi"][1] = [0.0, 1.0]; P["bc_T"][1] = [0.7, 0.0]
        nz, ny, nx = 1, 8, 8
        _compare_strip(oracle_mod, P, 10, 13)
        P = wl.base_params(8, 6, 7, grav=[1e-4, 0.0, -2e-4], **over)
        P["bc_f"][2] = ["wall", "wall"]; P["bc_g"][2] = ["zeroflux", "zeroflux"]; P["bc_s"][2] = ["dirichlet", "dirichlet"]
        P["bc_T"][2] = [1.0, 0.0]
        _compare(oracle_mod, P, 8, 14)


def _compare_strip(oracle_mod, P, steps, seed):
    """_compare on a state that is consistent with Dirichlet phi faces (a strip profile between the face values)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    shape = (P["nz"], P["ny"], P["nx"])
    y = (np.arange(P["ny"]) + .5)[None, :, None] / P["ny"]
    phi = 0.5 * (1 + np.tanh((y - 0.5) * 6)) + 0.005 * rng.uniform(-1, 1, shape)
    T = P["T_sat"] + rng.uniform(-0.3, 0.3, shape)
    u = 0.02 * rng.uniform(-1, 1, (3,) + shape); u[2] = 0
    p = 0.01 * rng.uniform(-1, 1, shape)
    o = oracle_mod.Oracle(P); o.init(phi, T, u, p)
    m = NPModel(P); m.init(phi, T, u, p)
    o.step(steps); m.step(steps)
    for a, b in zip(o.read_macro(), (m.phi, m.u, m.p, m.T)):
        assert np.abs(a - b).max() < 1e-13
    o.close()


def test_latent_heat_source_galilean_invariant_with_the_stencil_divergence(oracle_mod):
    """The pin of reading S5's u.grad(phi) term, repeated with div_scheme = "stencil": the latent-heat source is the material
    derivative of phi, so an evaporating slab carried by a uniform prescribed velocity evolves like the slab at rest,
    shifted.  Catches a stencil divergence with the wrong sign or missing from T or from S_i^s."""
    nx, ny, u0, steps = 128, 4, 0.01, 300
    P = wl.base_params(nx, ny, 1, rho_l=1.0, rho_g=1.0, sigma=0.0, prescribed_u=True, div_scheme="stencil")
    x = (np.arange(nx) + 0.5)[None, None, :] + np.zeros((1, ny, 1))
    phi0 = 0.5 * (1 - np.tanh(2 * (np.abs(x - 40.0) - 14.0) / P["W"]))
    T0 = P["T_sat"] + 0.3 * np.exp(-((x - 40.0) / 10.0) ** 2)

    def run(ux):
        u = np.zeros((3, 1, ny, nx)); u[0] = ux
        o = oracle_mod.Oracle(P); o.init(phi0, T0, u, None); o.step(steps)
        r = o.read_macro(); o.close()
        return r

    rest, moving = run(0.0), run(u0)
    k = int(round(u0 * steps))
    assert np.abs(rest[0] - phi0).max() > 0.01 and np.abs(rest[3] - T0).max() > 0.05
    assert np.abs(moving[0] - np.roll(rest[0], k, axis=2)).max() < 0.02
    assert np.abs(moving[3] - np.roll(rest[3], k, axis=2)).max() < 0.1


def test_stefan_interface_with_the_stencil_divergence(oracle_mod):
    """Config 2 (Stefan strip with the flow solved, open face): the stencil divergence sees the velocity jump of Eq.(11a)
    numerically instead of through phi m''' (1/rho_g - 1/rho_l); the interface must arrive where the product-rule run puts
    it (both within 1 % of each other after 3000 steps), and the liquid must still leave at the integrated mass source."""
    res = {}
    for scheme in ("product", "stencil"):
        P, I = wl.config2_stefan(nx=128, ny=4)
        P["div_scheme"] = scheme
        o = oracle_mod.Oracle(P); o.init(I["phi"], I["T"], None, None); o.step(3000)
        phi, u, _, _ = o.read_macro()
        _, _, pdot, _ = o.read_aux()
        o.close()
        row = phi[0, 0]
        i = int(np.where(row < 0.5)[0][0])
        xi = i - 0.5 + (row[i - 1] - 0.5) / (row[i - 1] - row[i]) + 0.5
        src = (P["rho_g"] * pdot[0, 0] * (1 / P["rho_g"] - 1 / P["rho_l"])).sum() * P["dx"]
        res[scheme] = (xi, u[0, 0, 0, 80:120] / src)
    assert abs(res["stencil"][0] / res["product"][0] - 1) < 0.01
    assert np.abs(res["stencil"][1] - 1).max() < 0.03
