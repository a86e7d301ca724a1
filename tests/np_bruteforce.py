"""Independent NumPy transcription of the coupled step, for brute-force pins of the C oracle on tiny grids.

Written from PAPER.md in a deliberately different style from oracle/lbm_oracle.c (and sharing nothing with
it or with the CUDA path): whole-array operations, np.roll streaming with masks for the boundary links,
ghost layers built with np.pad, lattices GENERATED from |e|^2 shells instead of typed tables, and the
collision in the paper's alternative form Eq.(C.11) instead of Eq.(C.10)/(25).
Population order therefore differs from the oracle's; compare by lattice vector (``vectors``).
"""
from __future__ import annotations

import itertools

import numpy as np

_SHELL_W = {
    "D2Q5": (2, {0: 1 / 3, 1: 1 / 6}),
    "D2Q9": (2, {0: 4 / 9, 1: 1 / 9, 2: 1 / 36}),
    "D3Q7": (3, {0: 1 / 4, 1: 1 / 8}),
    "D3Q19": (3, {0: 1 / 3, 1: 1 / 18, 2: 1 / 36}),
    "D3Q15": (3, {0: 2 / 9, 1: 1 / 9, 3: 1 / 72}),
}


def make_lattice(name):
    dim, shells = _SHELL_W[name]
    vecs, ws = [], []
    for v in itertools.product((-1, 0, 1), repeat=dim):
        n2 = sum(c * c for c in v)
        if n2 in shells:
            vecs.append(tuple(v) + (0,) * (3 - dim))
            ws.append(shells[n2])
    e = np.array(vecs, dtype=int)
    w = np.array(ws)
    assert abs(w.sum() - 1) < 1e-15
    e2 = float((w * e[:, 0] ** 2).sum())  # c_s^2 = e2 c^2
    return e, w, e2


class NPModel:
    def __init__(self, P):
        self.P = P
        self.shape = (P["nz"], P["ny"], P["nx"])
        self.ef, self.wf, self.e2f = make_lattice(P["lat_f"])
        self.eg, self.wg, self.e2g = make_lattice(P["lat_g"])
        self.es, self.ws, self.e2s = make_lattice(P["lat_s"])
        self.K = 1.5 * P["W"] * P["sigma"]      # Eq.(15b)
        self.H = 12.0 * P["sigma"] / P["W"]
        self.c = P["dx"] / P["dt"]

    # ---- ghost-padded fields (axis order x, y, z; array axes are (z, y, x)) ----------------------------
    @staticmethod
    def _ghosts(a, ax, depth, periodic):
        """(low ghosts, high ghosts) of array a along axis ax: periodic images, or mirror images in the faces (which sit
        half a cell outside the first / last node: ghost -1 <-> node 0, ghost -2 <-> node 1)."""
        n = a.shape[ax]
        if periodic:     # (modular: a 2D grid is one periodic layer thick in z)
            return (np.take(a, [k % n for k in range(-depth, 0)], axis=ax),
                    np.take(a, [k % n for k in range(n, n + depth)], axis=ax))
        first = np.take(a, range(depth), axis=ax)
        last = np.take(a, range(n - depth, n), axis=ax)
        return np.flip(first, axis=ax), np.flip(last, axis=ax)

    def _pad_phi(self, phi, depth=1):
        P = self.P
        a = phi
        for axis_phys, ax in ((0, 2), (1, 1), (2, 0)):
            kinds = P["bc_g"][axis_phys]
            glo, ghi = self._ghosts(a, ax, depth, kinds[0] == "periodic")
            if kinds[0] == "dirichlet":
                glo = 2.0 * P["bc_phi"][axis_phys][0] - glo
            if kinds[1] == "dirichlet":
                ghi = 2.0 * P["bc_phi"][axis_phys][1] - ghi
            a = np.concatenate([glo, a, ghi], axis=ax)
        return a

    def _pad_u(self, ua):
        """One velocity component with one ghost layer (reading S17): periodic image; no-slip wall: odd reflection (zero on
        the wall); open face: even reflection."""
        P = self.P
        a = ua
        for axis_phys, ax in ((0, 2), (1, 1), (2, 0)):
            kinds = P["bc_f"][axis_phys]
            glo, ghi = self._ghosts(a, ax, 1, kinds[0] == "periodic")
            if kinds[0] == "wall":
                glo = -glo
            if kinds[1] == "wall":
                ghi = -ghi
            a = np.concatenate([glo, a, ghi], axis=ax)
        return a

    def derive(self, phi):
        """grad phi Eq.(35a,b), lap phi Eq.(36a,b) on the NS lattice; the directional derivative inside
        Eq.(35b) central (35a) or one of the biased differences of PAPER.md:318."""
        P = self.P
        nz, ny, nx = self.shape
        scheme = P.get("grad_scheme", "central")
        pad = self._pad_phi(phi, 2)

        def sh(v):
            return pad[2 + v[2]:2 + v[2] + nz, 2 + v[1]:2 + v[1] + ny, 2 + v[0]:2 + v[0] + nx]

        grad = np.zeros((3,) + self.shape)
        lap = np.zeros(self.shape)
        for v, w in zip(self.ef, self.wf):
            if not v.any():
                continue
            plus, minus = sh(v), sh(-v)
            if scheme == "central":
                dd = (plus - minus) / (2 * P["dx"])
            elif scheme == "biased1":
                dd = (plus - phi) / P["dx"]
            else:
                dd = (4 * plus - sh(2 * v) - 3 * phi) / (2 * P["dx"])
            for a in range(3):
                grad[a] += w * v[a] * dd
            lap += w * (plus - 2 * phi + minus) / P["dx"] ** 2
        return grad / self.e2f, lap / self.e2f

    def div_uphi(self, u, phi, grad, mdot):
        """div(u phi): product rule with Eq.(11a) (reading S5) or the directional-derivative stencil on u phi (S17)."""
        P = self.P
        if P.get("div_scheme", "product") == "product":
            return (u * grad).sum(axis=0) + phi * mdot * (1 / P["rho_g"] - 1 / P["rho_l"])
        nz, ny, nx = self.shape
        pphi = self._pad_phi(phi, 1)
        flux = [self._pad_u(u[a]) * pphi for a in range(3)]
        D = np.zeros(self.shape)
        for v, w in zip(self.ef, self.wf):
            for a in range(3):
                if v[a]:
                    D += w * v[a] * flux[a][1 + v[2]:1 + v[2] + nz, 1 + v[1]:1 + v[1] + ny, 1 + v[0]:1 + v[0] + nx]
        return D / (self.e2f * P["dx"])

    def pdot_of(self, phi, T):
        P = self.P
        if not P["phase_change"]:
            return np.zeros_like(phi)
        alpha = phi * P["alpha_g"] + (1 - phi) * P["alpha_l"]
        theta = P["Cp"] * (T - P["T_sat"]) / P["L_latent"]
        return 4 * alpha / (P["A"] * P["W"] ** 2) * (theta - P["theta_I"]) * phi * (1 - phi)   # Eq.(18)

    def _closures(self, phi, grad, lap):
        P = self.P
        rho = phi * P["rho_g"] + (1 - phi) * P["rho_l"]
        mu = 4 * self.H * phi * (phi - 1) * (phi - 0.5) - self.K * lap                          # Eq.(14)
        g = np.array(P["grav"]).reshape(3, 1, 1, 1)
        fb = np.array(P.get("force", (0.0, 0.0, 0.0))).reshape(3, 1, 1, 1)
        F = mu * grad + (rho - P["rho_l"]) * g + fb                                              # Eq.(12),(13), G6
        grho = (P["rho_g"] - P["rho_l"]) * grad
        return rho, F, grho

    @staticmethod
    def _gamma(e, w, c, cs2, u):
        cu = c * np.tensordot(e.astype(float), u, axes=(1, 0))           # (Q, z, y, x)
        uu = (u * u).sum(axis=0)
        return w[:, None, None, None] * (1 + cu / cs2 + cu ** 2 / (2 * cs2 ** 2) - uu / (2 * cs2))   # Eq.(27d)

    def eq_sources(self):
        P = self.P
        c, dt = self.c, P["dt"]
        phi, T, p, u = self.phi, self.T, self.p, self.u
        grad, lap = self.grad, self.lap
        rho, F, grho = self._closures(phi, grad, lap)
        nu = P["nu_l"] * P["nu_g"] / (phi * P["nu_l"] + (1 - phi) * P["nu_g"])                   # Eq.(1b)
        alpha = phi * P["alpha_g"] + (1 - phi) * P["alpha_l"]
        nrm = grad / np.sqrt((grad ** 2).sum(axis=0) + P["eps_n"] ** 2)
        drho = 1 / P["rho_g"] - 1 / P["rho_l"]
        mdot = P["rho_g"] * self.pdot
        D = self.div_uphi(u, phi, grad, mdot)
        out = {}
        # NS
        cs2 = self.e2f * c * c
        G = self._gamma(self.ef, self.wf, c, cs2, u)
        W_ = self.wf[:, None, None, None]
        feq = W_ * p + rho * cs2 * (G - W_)                                                      # Eq.(26b)
        S = W_ * rho * cs2 * mdot * drho                                                         # Eq.(27c)
        for a in range(3):
            ca = c * self.ef[:, a].astype(float)[:, None, None, None]
            S = S + (ca - u[a]) * ((G - W_) * grho[a] * cs2 + G * F[a])                          # Eq.(27b)
        out["f"] = (feq, S, nu / (cs2 * dt))
        # CAC, modified-equilibrium form Eq.(31b)
        cs2 = self.e2g * c * c
        G = self._gamma(self.eg, self.wg, c, cs2, u)
        W_ = self.wg[:, None, None, None]
        cn = c * np.tensordot(self.eg.astype(float), nrm, axes=(1, 0))
        geq = phi * G + P["M"] * 4 / P["W"] * phi * (1 - phi) * W_ * cn / cs2
        out["g"] = (geq, W_ * self.pdot, np.full(self.shape, P["M"] / (cs2 * dt)))
        # heat
        cs2 = self.e2s * c * c
        G = self._gamma(self.es, self.ws, c, cs2, u)
        W_ = self.ws[:, None, None, None]
        S = -W_ * (P["L_latent"] / P["Cp"]) * (self.dtphi + D) if P["latent_heat"] else 0 * G    # Eq.(33c,d), G2
        out["s"] = (T * G, S, alpha / (cs2 * dt))
        return out

    def init(self, phi, T=None, u=None, p=None):
        P = self.P
        self.phi = np.array(phi, dtype=float)
        self.T = np.full(self.shape, P["T_sat"]) if T is None else np.array(T, dtype=float)
        self.u = np.zeros((3,) + self.shape) if u is None else np.array(u, dtype=float)
        self.p = np.zeros(self.shape) if p is None else np.array(p, dtype=float)
        self.dtphi = np.zeros(self.shape)
        self.pdot = self.pdot_of(self.phi, self.T)
        self.grad, self.lap = self.derive(self.phi)
        t = self.eq_sources()
        self.pops = {k: t[k][0] - 0.5 * P["dt"] * t[k][1] for k in "fgs"}                        # Eq.(24)

    def _stream(self, post, e, w, kinds, vals, is_f):
        """Pull streaming: roll, then overwrite the links that cross a non-periodic face (S8)."""
        nz, ny, nx = self.shape
        lens = (nx, ny, nz)
        axes = (2, 1, 0)
        coords = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
        coord = {0: coords[2], 1: coords[1], 2: coords[0]}
        opp = [int(np.where((e == -v).all(axis=1))[0][0]) for v in e]
        out = np.empty_like(post)
        for i, v in enumerate(e):
            a = post[i]
            for ax in range(3):
                if v[ax]:
                    a = np.roll(a, v[ax], axis=axes[ax])
            decided = np.zeros(self.shape, dtype=bool)
            for ax in range(3):               # lowest axis decides
                if not v[ax] or kinds[ax][0] == "periodic":
                    continue
                side = 0 if v[ax] > 0 else 1  # source x - e is below 0 when e > 0
                edge = coord[ax] == (0 if side == 0 else lens[ax] - 1)
                m = edge & ~decided
                kind = kinds[ax][side]
                back = post[opp[i]]
                if kind in ("wall", "zeroflux"):
                    a = np.where(m, back, a)
                else:                          # "open" (f) or "dirichlet" (g, s): anti-bounce-back
                    a = np.where(m, -back + 2 * w[i] * vals[ax][side], a)
                decided |= edge
            out[i] = a
        return out

    def step(self, n=1):
        P = self.P
        dt, c = P["dt"], self.c
        for _ in range(n):
            t = self.eq_sources()
            post = {}
            for k in "fgs":
                eq, S, tau = t[k]
                om = 1 / (tau + 0.5)
                post[k] = self.pops[k] - om * (self.pops[k] - eq) + tau * om * dt * S              # Eq.(C.11)
            self.pops["f"] = self._stream(post["f"], self.ef, self.wf, P["bc_f"], P["bc_p"], True)
            self.pops["g"] = self._stream(post["g"], self.eg, self.wg, P["bc_g"], P["bc_phi"], False)
            self.pops["s"] = self._stream(post["s"], self.es, self.ws, P["bc_s"], P["bc_T"], False)
            # moments (S3 order)
            phinew = self.pops["g"].sum(axis=0) + 0.5 * dt * self.pdot                             # Eq.(32)
            self.dtphi = (phinew - self.phi) / dt
            self.phi = phinew
            self.grad, self.lap = self.derive(self.phi)
            rho, F, grho = self._closures(self.phi, self.grad, self.lap)
            cs2 = self.e2f * c * c
            m1 = c * np.tensordot(self.ef.astype(float).T, self.pops["f"], axes=(1, 0))
            if not P.get("prescribed_u", False):
                self.u = (m1 / cs2 + 0.5 * dt * F) / rho                                           # Eq.(28a)
            drho = 1 / P["rho_g"] - 1 / P["rho_l"]
            mdot = P["rho_g"] * self.pdot
            D = self.div_uphi(self.u, self.phi, self.grad, mdot)
            self.T = self.pops["s"].sum(axis=0)
            if P["latent_heat"]:
                self.T = self.T - 0.5 * dt * (P["L_latent"] / P["Cp"]) * (self.dtphi + D)          # Eq.(34)
            self.p = self.pops["f"].sum(axis=0) + 0.5 * dt * (
                cs2 * (self.u * grho).sum(axis=0) + rho * cs2 * mdot * drho)                       # Eq.(28b)
            self.pdot = self.pdot_of(self.phi, self.T)

    def vectors(self, which):
        return {"f": self.ef, "g": self.eg, "s": self.es}[which]
