"""Closed forms the paper fixes, used to pin the oracle (no lattice Boltzmann code here)."""
from __future__ import annotations

import math

from scipy.optimize import brentq
from scipy.special import erf, erfc


def stefan_xi_two_phase(theta_w, theta_inf, theta_I, alpha_l, alpha_g):
    """Root of the transcendental Eq.(41d) with the right-hand side read as
    xi sqrt(pi) / (theta_I - theta_w) (reading G5; equals the printed -xi sqrt(pi)/theta_w when theta_I = 0)."""
    r = alpha_l / alpha_g

    def fun(xi):
        return (math.exp(-xi * xi) / erf(xi)
                + math.sqrt(1.0 / r) * (theta_I - theta_inf) / (theta_I - theta_w)
                * math.exp(-xi * xi * r) / erfc(xi * math.sqrt(r))
                - xi * math.sqrt(math.pi) / (theta_I - theta_w))

    return brentq(fun, 1e-6, 3.0, xtol=1e-14)


def stefan_xi_printed_rhs(theta_w, theta_inf, theta_I, alpha_l, alpha_g):
    """Same with the right-hand side exactly as printed, -xi sqrt(pi)/theta_w."""
    r = alpha_l / alpha_g

    def fun(xi):
        return (math.exp(-xi * xi) / erf(xi)
                + math.sqrt(1.0 / r) * (theta_I - theta_inf) / (theta_I - theta_w)
                * math.exp(-xi * xi * r) / erfc(xi * math.sqrt(r))
                + xi * math.sqrt(math.pi) / theta_w)

    return brentq(fun, 1e-6, 3.0, xtol=1e-14)


def stefan_xi_one_phase(St):
    """xi exp(xi^2) erf(xi) = St / sqrt(pi): classical one-phase Stefan problem (ref. [66] of the paper)."""
    return brentq(lambda xi: xi * math.exp(xi * xi) * erf(xi) - St / math.sqrt(math.pi), 1e-9, 3.0, xtol=1e-14)


def film_boiling_numbers(rho_l, rho_g, nu_g, alpha_g, sigma, g_y, theta_w):
    """lambda_s, lambda_c, t_s, Gr, Pr, Ja of Eq.(43) and PAPER.md:529-535."""
    lam_s = math.sqrt(sigma / ((rho_l - rho_g) * g_y))
    return dict(lambda_s=lam_s, lambda_c=2 * math.pi * lam_s, t_s=math.sqrt(lam_s / g_y),
                Gr=rho_g * g_y * (rho_l - rho_g) * lam_s ** 3 / (rho_g ** 2 * nu_g ** 2),
                Pr=nu_g / alpha_g, Ja=theta_w)
