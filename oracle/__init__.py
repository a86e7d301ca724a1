"""CPU oracle binding -- TEST INFRASTRUCTURE ONLY.

Loads ``oracle/liboracle.so`` (built from ``oracle/lbm_oracle.c`` with gcc, no CUDA) through ctypes.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package; the product package ``paper_2003_06342_b200`` never does.

The parameter dictionary accepted by :class:`Oracle` is the plain description produced by
``paper_2003_06342_b200.workloads`` (names of the paper's symbols; no arithmetic of the method).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

LATTICES = {"D2Q5": 0, "D2Q9": 1, "D3Q7": 2, "D3Q19": 3, "D3Q15": 4}
LATTICE_Q = {"D2Q5": 5, "D2Q9": 9, "D3Q7": 7, "D3Q19": 19, "D3Q15": 15}
F_KINDS = {"periodic": 0, "wall": 1, "open": 2}
S_KINDS = {"periodic": 0, "zeroflux": 1, "dirichlet": 2}
FLAG_PHASE_CHANGE = 1
FLAG_LATENT_HEAT = 2
FLAG_PRESCRIBED_U = 4
CAC_MODIFIED_EQ = 0
CAC_SOURCE = 1
POPS_POSTCOLLISION = 0
POPS_STREAMED = 1
GRAD_SCHEMES = {"central": 0, "biased1": 1, "biased2": 2}
DIV_SCHEMES = {"product": 0, "stencil": 1}                  # DESIGN.md readings S5 / S17


class _Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("lat_f", C.c_int), ("lat_g", C.c_int), ("lat_s", C.c_int),
        ("bc_f", (C.c_int * 2) * 3), ("bc_g", (C.c_int * 2) * 3), ("bc_s", (C.c_int * 2) * 3),
        ("bc_phi", (C.c_double * 2) * 3), ("bc_T", (C.c_double * 2) * 3), ("bc_p", (C.c_double * 2) * 3),
        ("dx", C.c_double), ("dt", C.c_double),
        ("rho_l", C.c_double), ("rho_g", C.c_double), ("nu_l", C.c_double), ("nu_g", C.c_double),
        ("sigma", C.c_double), ("W", C.c_double), ("M", C.c_double),
        ("grav", C.c_double * 3), ("force", C.c_double * 3),
        ("alpha_l", C.c_double), ("alpha_g", C.c_double),
        ("L_latent", C.c_double), ("Cp", C.c_double), ("T_sat", C.c_double), ("theta_I", C.c_double),
        ("A", C.c_double), ("eps_n", C.c_double),
        ("flags", C.c_uint),
        ("grad_scheme", C.c_int), ("div_scheme", C.c_int),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (``-O2 -ffp-contract=off -fopenmp``); returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(
            os.path.getmtime(_SRC), os.path.getmtime(os.path.join(_HERE, "lbm_oracle.h"))):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-Wall", "-Wextra", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.POINTER(_Params)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_init.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.oracle_step.argtypes = [C.c_void_p, C.c_int]
        L.oracle_read_macro.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.oracle_read_pops.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.oracle_read_aux.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.oracle_read_div.argtypes = [C.c_void_p, dp]
        L.oracle_set_cac_form.argtypes = [C.c_void_p, C.c_int]
        L.oracle_set_velocity.argtypes = [C.c_void_p, dp]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_lattice.argtypes = [C.c_int, C.POINTER(C.c_int), dp, dp]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def fill_params(P: dict) -> _Params:
    s = _Params()
    s.nx, s.ny, s.nz = int(P["nx"]), int(P["ny"]), int(P.get("nz", 1))
    s.lat_f, s.lat_g, s.lat_s = (LATTICES[P[k]] for k in ("lat_f", "lat_g", "lat_s"))
    for a in range(3):
        for side in range(2):
            s.bc_f[a][side] = F_KINDS[P["bc_f"][a][side]]
            s.bc_g[a][side] = S_KINDS[P["bc_g"][a][side]]
            s.bc_s[a][side] = S_KINDS[P["bc_s"][a][side]]
            s.bc_phi[a][side] = float(P["bc_phi"][a][side])
            s.bc_T[a][side] = float(P["bc_T"][a][side])
            s.bc_p[a][side] = float(P["bc_p"][a][side])
    for k in ("dx", "dt", "rho_l", "rho_g", "nu_l", "nu_g", "sigma", "W", "M", "alpha_l", "alpha_g",
              "L_latent", "Cp", "T_sat", "theta_I", "A", "eps_n"):
        setattr(s, k, float(P[k]))
    for a in range(3):
        s.grav[a] = float(P["grav"][a])
        s.force[a] = float(P.get("force", (0.0, 0.0, 0.0))[a])
    s.flags = (FLAG_PHASE_CHANGE if P["phase_change"] else 0) | (FLAG_LATENT_HEAT if P["latent_heat"] else 0) | (
        FLAG_PRESCRIBED_U if P.get("prescribed_u", False) else 0)
    s.grad_scheme = GRAD_SCHEMES[P.get("grad_scheme", "central")]
    s.div_scheme = DIV_SCHEMES[P.get("div_scheme", "product")]
    return s


def lattice(name: str):
    """(e[Q,3] int, w[Q], e2) of the oracle's lattice tables."""
    Q = LATTICE_Q[name]
    e = np.zeros((Q, 3), dtype=np.int32)
    w = np.zeros(Q)
    e2 = C.c_double()
    q = lib().oracle_lattice(LATTICES[name], e.ctypes.data_as(C.POINTER(C.c_int)), _ptr(w), C.byref(e2))
    assert q == Q
    return e, w, e2.value


def num_threads() -> int:
    return int(lib().oracle_num_threads())


class Oracle:
    """Thin handle on one oracle context.  Arrays are float64, shape (nz, ny, nx) (u: (3, nz, ny, nx))."""

    def __init__(self, P: dict):
        self.P = dict(P)
        self.shape = (int(P.get("nz", 1)), int(P["ny"]), int(P["nx"]))
        self.N = self.shape[0] * self.shape[1] * self.shape[2]
        self.Q = tuple(LATTICE_Q[P[k]] for k in ("lat_f", "lat_g", "lat_s"))
        self._s = fill_params(P)
        self._h = lib().oracle_create(C.byref(self._s))
        if not self._h:
            raise ValueError("oracle_create rejected the parameters")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _arr(a, shape):
        if a is None:
            return None
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == shape, (a.shape, shape)
        return a

    def init(self, phi, T=None, u=None, p=None):
        phi = self._arr(phi, self.shape)
        T = self._arr(T, self.shape)
        u = self._arr(u, (3,) + self.shape)
        p = self._arr(p, self.shape)
        rc = lib().oracle_init(self._h, _ptr(phi), _ptr(T), _ptr(u), _ptr(p))
        assert rc == 0

    def step(self, n=1):
        assert lib().oracle_step(self._h, int(n)) == 0

    def set_cac_form(self, form):
        lib().oracle_set_cac_form(self._h, int(form))

    def set_velocity(self, u):
        """Prescribed-velocity mode: u of the next time level."""
        u = self._arr(u, (3,) + self.shape)
        assert lib().oracle_set_velocity(self._h, _ptr(u)) == 0

    def read_macro(self):
        phi = np.empty(self.shape)
        u = np.empty((3,) + self.shape)
        p = np.empty(self.shape)
        T = np.empty(self.shape)
        assert lib().oracle_read_macro(self._h, _ptr(phi), _ptr(u), _ptr(p), _ptr(T)) == 0
        return phi, u, p, T

    def read_pops(self, which, stage=POPS_STREAMED):
        out = np.empty((self.Q[which],) + self.shape)
        assert lib().oracle_read_pops(self._h, int(which), int(stage), _ptr(out)) == 0
        return out

    def read_div(self):
        """div(u phi) of the current level by the stencil (div_scheme "stencil" only)."""
        out = np.empty(self.shape)
        assert lib().oracle_read_div(self._h, _ptr(out)) == 0
        return out

    def read_aux(self):
        grad = np.empty((3,) + self.shape)
        lap = np.empty(self.shape)
        pdot = np.empty(self.shape)
        dtphi = np.empty(self.shape)
        assert lib().oracle_read_aux(self._h, _ptr(grad), _ptr(lap), _ptr(pdot), _ptr(dtphi)) == 0
        return grad, lap, pdot, dtphi
