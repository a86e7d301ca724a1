"""Thin Python binding of the C ABI in ``include/lbm.h`` (argument marshalling only).

Same names as the C calls: :func:`lbm_workspace_bytes`, :class:`LBM` with ``init / step / read_macro / read_pops /
sync / destroy``.  PyTorch is used for the device allocation and the CUDA stream only; every step of the path runs
in the library's kernels.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblbm_b200.so")

LATTICES = {"D2Q5": 0, "D2Q9": 1, "D3Q7": 2, "D3Q19": 3, "D3Q15": 4}
LATTICE_Q = {"D2Q5": 5, "D2Q9": 9, "D3Q7": 7, "D3Q19": 19, "D3Q15": 15}
F_KINDS = {"periodic": 0, "wall": 1, "open": 2}
S_KINDS = {"periodic": 0, "zeroflux": 1, "dirichlet": 2}
GRAD_SCHEMES = {"central": 0, "biased1": 1, "biased2": 2}   # lbm_params.grad_scheme (LBM_GRAD_*)
DIV_SCHEMES = {"product": 0, "stencil": 1}                  # lbm_params.div_scheme (LBM_DIV_*)
FLAG_PHASE_CHANGE = 1
FLAG_LATENT_HEAT = 2
FLAG_PRESCRIBED_U = 4
# kernel selection (include/lbm.h): speed only, never the method
FLAG_POPS_GATHER, FLAG_POPS_STAGED, FLAG_PHI_LDG, FLAG_NO_GRAPH, FLAG_NO_PDL, FLAG_ONE_NODE = 16, 32, 64, 128, 256, 512
KERNEL_FLAGS = {"pops_gather": FLAG_POPS_GATHER, "pops_staged": FLAG_POPS_STAGED,
                "phi_ldg": FLAG_PHI_LDG, "no_graph": FLAG_NO_GRAPH, "no_pdl": FLAG_NO_PDL, "one_node": FLAG_ONE_NODE}
POPS_F, POPS_G, POPS_S = 0, 1, 2
STAGE_POSTCOLLISION, STAGE_STREAMED = 0, 1
HALO_PHI, HALO_POPS = 0, 1
NOALLOC_SCRATCH_BYTES = 8 << 20

EXPORTS = ["lbm_workspace_bytes", "lbm_create", "lbm_init", "lbm_step", "lbm_set_velocity", "lbm_step_phase", "lbm_step_layers", "lbm_set_stream", "lbm_halo_bytes", "lbm_halo_pack", "lbm_halo_unpack", "lbm_halo_push", "lbm_halo_push_mapped", "lbm_stream_signal", "lbm_stream_wait", "lbm_read_macro", "lbm_read_pops", "lbm_read_pops_noalloc",
           "lbm_sync", "lbm_check_finite", "lbm_state_bytes", "lbm_save_state", "lbm_load_state", "lbm_set_timing", "lbm_kernel_times", "lbm_note_replay", "lbm_step_count", "lbm_launch_count", "lbm_variant", "lbm_last_cuda_error", "lbm_strerror",
           "lbm_destroy"]


class lbm_params(C.Structure):
    """Mirror of ``struct lbm_params`` (include/lbm.h)."""
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("lat_f", C.c_int), ("lat_g", C.c_int), ("lat_s", C.c_int),
        ("precision", C.c_int),
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
        ("halo", C.c_int * 2),
        ("grad_scheme", C.c_int), ("div_scheme", C.c_int),
    ]


class LBMError(RuntimeError):
    pass


_lib = None


def load_library():
    """dlopen the in-tree C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise LBMError("%s is missing: run `python -m paper_2003_06342_b200.build` (there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        L.lbm_workspace_bytes.restype = C.c_size_t
        L.lbm_workspace_bytes.argtypes = [C.POINTER(lbm_params)]
        L.lbm_create.argtypes = [C.POINTER(lbm_params), C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        L.lbm_init.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.lbm_step.argtypes = [C.c_void_p, C.c_int]
        L.lbm_set_velocity.argtypes = [C.c_void_p, C.c_void_p]
        L.lbm_step_phase.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.lbm_step_layers.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        L.lbm_set_stream.argtypes = [C.c_void_p, C.c_void_p]
        L.lbm_halo_bytes.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_size_t)]
        L.lbm_halo_pack.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.lbm_halo_unpack.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.lbm_halo_push.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.lbm_halo_push_mapped.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(lbm_params), C.c_void_p]
        L.lbm_stream_signal.argtypes = [C.c_void_p, C.c_void_p, C.c_uint]
        L.lbm_stream_wait.argtypes = [C.c_void_p, C.c_void_p, C.c_uint]
        L.lbm_read_macro.argtypes = [C.c_void_p] + [C.c_void_p] * 4
        L.lbm_read_pops.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.lbm_read_pops_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.lbm_sync.argtypes = [C.c_void_p]
        L.lbm_check_finite.argtypes = [C.c_void_p, C.POINTER(C.c_longlong)]
        L.lbm_state_bytes.restype = C.c_size_t
        L.lbm_state_bytes.argtypes = [C.c_void_p]
        L.lbm_save_state.argtypes = [C.c_void_p, C.c_void_p]
        L.lbm_load_state.argtypes = [C.c_void_p, C.c_void_p]
        L.lbm_set_timing.argtypes = [C.c_void_p, C.c_int]
        L.lbm_kernel_times.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.lbm_note_replay.argtypes = [C.c_void_p, C.c_longlong, C.c_longlong]
        L.lbm_step_count.restype = C.c_longlong
        L.lbm_step_count.argtypes = [C.c_void_p]
        L.lbm_launch_count.restype = C.c_longlong
        L.lbm_launch_count.argtypes = [C.c_void_p]
        L.lbm_variant.restype = C.c_char_p
        L.lbm_variant.argtypes = [C.c_void_p]
        L.lbm_last_cuda_error.restype = C.c_int
        L.lbm_strerror.restype = C.c_char_p
        L.lbm_strerror.argtypes = [C.c_int]
        L.lbm_destroy.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def make_params(P: dict, precision: int = 64) -> lbm_params:
    s = lbm_params()
    s.nx, s.ny, s.nz = int(P["nx"]), int(P["ny"]), int(P.get("nz", 1))
    s.lat_f, s.lat_g, s.lat_s = (LATTICES[P[k]] for k in ("lat_f", "lat_g", "lat_s"))
    s.precision = int(precision)
    for a in range(3):
        for side in range(2):
            s.bc_f[a][side] = F_KINDS[P["bc_f"][a][side]]
            s.bc_g[a][side] = S_KINDS[P["bc_g"][a][side]]
            s.bc_s[a][side] = S_KINDS[P["bc_s"][a][side]]
            s.bc_phi[a][side] = float(P["bc_phi"][a][side])
            s.bc_T[a][side] = float(P["bc_T"][a][side])
            s.bc_p[a][side] = float(P["bc_p"][a][side])
        s.grav[a] = float(P["grav"][a])
        s.force[a] = float(P.get("force", (0.0, 0.0, 0.0))[a])
    for k in ("dx", "dt", "rho_l", "rho_g", "nu_l", "nu_g", "sigma", "W", "M", "alpha_l", "alpha_g",
              "L_latent", "Cp", "T_sat", "theta_I", "A", "eps_n"):
        setattr(s, k, float(P[k]))
    s.flags = (FLAG_PHASE_CHANGE if P["phase_change"] else 0) | (FLAG_LATENT_HEAT if P["latent_heat"] else 0) | (
        FLAG_PRESCRIBED_U if P.get("prescribed_u", False) else 0)
    for name in P.get("kernels", ()):        # e.g. P["kernels"] = ("pops_gather",): force a plainer kernel variant
        s.flags |= KERNEL_FLAGS[name]
    halo = P.get("halo", (0, 0))
    s.halo[0], s.halo[1] = int(halo[0]), int(halo[1])
    s.grad_scheme = GRAD_SCHEMES[P.get("grad_scheme", "central")]     # model variants (include/lbm.h)
    s.div_scheme = DIV_SCHEMES[P.get("div_scheme", "product")]
    return s


def lbm_strerror(code: int) -> str:
    return load_library().lbm_strerror(int(code)).decode()


def _check(rc: int, what: str):
    if rc != 0:
        L = load_library()
        raise LBMError("%s failed: %s (code %d, cuda error %d)" % (what, lbm_strerror(rc), rc, L.lbm_last_cuda_error()))


def lbm_workspace_bytes(P: dict, precision: int = 64) -> int:
    s = make_params(P, precision)
    return int(load_library().lbm_workspace_bytes(C.byref(s)))


def _host_ptr(a, dtype, shape, name, output=False):
    """Pointer to a numpy array or a torch tensor (CPU, pinned or not, or CUDA: the library copies with unified
    addressing), contiguous, right dtype/shape.  Inputs may be converted (a temporary copy); an ``output`` array is
    written in place, so a wrong dtype, shape or layout raises instead."""
    if a is None:
        return None, None
    if isinstance(a, np.ndarray):
        if output:
            if a.dtype != dtype or not a.flags["C_CONTIGUOUS"] or not a.flags["WRITEABLE"] or tuple(a.shape) != tuple(shape):
                raise ValueError("%s: output must be a writable C-contiguous %s array of shape %s" % (name, np.dtype(dtype), shape))
            return a.ctypes.data, a
        b = np.ascontiguousarray(a, dtype=dtype)
        if tuple(b.shape) != tuple(shape):
            raise ValueError("%s: shape %s, expected %s" % (name, b.shape, shape))
        return b.ctypes.data, b
    import torch
    if isinstance(a, torch.Tensor):
        if not a.is_contiguous() or tuple(a.shape) != tuple(shape):
            raise ValueError("%s: need a contiguous tensor of shape %s" % (name, shape))
        want = torch.float64 if dtype == np.float64 else torch.float32
        if a.dtype != want:
            raise ValueError("%s: dtype %s, expected %s" % (name, a.dtype, want))
        return a.data_ptr(), a
    raise TypeError("%s: numpy array or torch tensor expected" % name)


class LBM:
    """One simulation context on the current CUDA device and stream."""

    def __init__(self, P: dict, precision: int = 64, stream=None, workspace=None):
        import torch
        if not torch.cuda.is_available():
            raise LBMError("no CUDA device: the library has no CPU path")
        self._L = load_library()
        self.P = dict(P)
        self.precision = int(precision)
        self.dtype = np.float64 if precision == 64 else np.float32
        self.shape = (int(P.get("nz", 1)), int(P["ny"]), int(P["nx"]))
        self.N = self.shape[0] * self.shape[1] * self.shape[2]
        self.Q = tuple(LATTICE_Q[P[k]] for k in ("lat_f", "lat_g", "lat_s"))
        self._params = make_params(P, precision)
        nbytes = int(self._L.lbm_workspace_bytes(C.byref(self._params)))
        if nbytes == 0:
            raise LBMError("lbm_workspace_bytes rejected the parameters")
        self.workspace_bytes = nbytes
        # device memory is allocated by torch and lent to the library (torch allocations are 512-byte aligned)
        # (or by the caller: ``workspace`` = a uint8 CUDA tensor of at least ``lbm_workspace_bytes`` bytes, 256-byte aligned)
        if workspace is None:
            workspace = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        elif workspace.dtype != torch.uint8 or workspace.device.type != "cuda" or not workspace.is_contiguous() or workspace.numel() < nbytes:
            raise ValueError("workspace: contiguous uint8 CUDA tensor of at least %d bytes expected" % nbytes)
        self._ws = workspace
        # A stream of the context's own unless the caller gives one: every call below is enqueued there, and the CUDA-graph
        # replay of small grids needs a stream that can be captured (the legacy default stream cannot).
        self._stream = stream if stream is not None else torch.cuda.Stream()
        h = C.c_void_p()
        _check(self._L.lbm_create(C.byref(self._params), C.c_void_p(self._ws.data_ptr()), nbytes,
                                  C.c_void_p(self._stream.cuda_stream), C.byref(h)), "lbm_create")
        self._h = h

    # -- the calls of include/lbm.h --------------------------------------------------------------------------
    def init(self, phi, T=None, u=None, p=None):
        keep = []
        ptrs = []
        for a, shape, name in ((phi, self.shape, "phi"), (T, self.shape, "T"), (u, (3,) + self.shape, "u"),
                               (p, self.shape, "p")):
            ptr, k = _host_ptr(a, self.dtype, shape, name)
            ptrs.append(C.c_void_p(ptr) if ptr is not None else None)
            keep.append(k)
        _check(self._L.lbm_init(self._h, *ptrs), "lbm_init")

    def step(self, n: int = 1):
        _check(self._L.lbm_step(self._h, int(n)), "lbm_step")

    # slab contexts (P["halo"]): the two phases of a step and the ghost-layer buffers, see include/lbm.h
    def step_phase(self, phase: int, store_macros: bool = False):
        _check(self._L.lbm_step_phase(self._h, int(phase), 1 if store_macros else 0), "lbm_step_phase")

    def step_layers(self, phase: int, first: int, count: int, store_macros: bool = False, last: bool = False):
        _check(self._L.lbm_step_layers(self._h, int(phase), int(first), int(count), 1 if store_macros else 0, 1 if last else 0),
               "lbm_step_layers")

    def set_stream(self, stream):
        """Enqueue the following calls on ``stream`` (a torch.cuda.Stream); the caller orders the streams with events."""
        _check(self._L.lbm_set_stream(self._h, C.c_void_p(stream.cuda_stream)), "lbm_set_stream")
        self._stream = stream

    def halo_bytes(self, what: int) -> int:
        n = C.c_size_t()
        _check(self._L.lbm_halo_bytes(self._h, int(what), C.byref(n)), "lbm_halo_bytes")
        return int(n.value)

    def _dev_buf(self, what, buf):
        if buf.device.type != "cuda" or not buf.is_contiguous() or buf.numel() * buf.element_size() < self.halo_bytes(what):
            raise ValueError("halo buffer: contiguous CUDA tensor of at least %d bytes expected" % self.halo_bytes(what))
        return C.c_void_p(buf.data_ptr())

    def halo_pack(self, what: int, side: int, buf):
        _check(self._L.lbm_halo_pack(self._h, int(what), int(side), self._dev_buf(what, buf)), "lbm_halo_pack")

    def halo_unpack(self, what: int, side: int, buf):
        _check(self._L.lbm_halo_unpack(self._h, int(what), int(side), self._dev_buf(what, buf)), "lbm_halo_unpack")

    def halo_push(self, what: int, side: int, peer: "LBM"):
        """lbm_halo_push: this slab's boundary layer of ``side`` straight into the opposite ghost layer of ``peer`` (one launch)."""
        _check(self._L.lbm_halo_push(self._h, int(what), int(side), peer._h), "lbm_halo_push")

    def halo_push_mapped(self, what: int, side: int, peer_params: dict, peer_workspace_ptr: int):
        """lbm_halo_push_mapped: as halo_push, for a neighbour known by its parameters and its (peer-mapped) workspace pointer."""
        s = make_params(peer_params, self.precision)
        _check(self._L.lbm_halo_push_mapped(self._h, int(what), int(side), C.byref(s), C.c_void_p(int(peer_workspace_ptr))),
               "lbm_halo_push_mapped")

    def stream_signal(self, flag_ptr: int, value: int):
        """lbm_stream_signal: write ``value`` to the 32-bit device word at ``flag_ptr`` after what this context has enqueued so far."""
        _check(self._L.lbm_stream_signal(self._h, C.c_void_p(int(flag_ptr)), int(value) & 0xFFFFFFFF), "lbm_stream_signal")

    def stream_wait(self, flag_ptr: int, value: int):
        """lbm_stream_wait: hold this context's stream until the 32-bit device word at ``flag_ptr`` is >= ``value``."""
        _check(self._L.lbm_stream_wait(self._h, C.c_void_p(int(flag_ptr)), int(value) & 0xFFFFFFFF), "lbm_stream_wait")

    def set_velocity(self, u):
        ptr, keep = _host_ptr(u, self.dtype, (3,) + self.shape, "u")
        _check(self._L.lbm_set_velocity(self._h, C.c_void_p(ptr)), "lbm_set_velocity")

    def read_macro(self, out=None):
        """Returns (phi, u, p, T) as numpy arrays; ``out`` may give preallocated host arrays/tensors (pinned)."""
        if out is None:
            out = (np.empty(self.shape, self.dtype), np.empty((3,) + self.shape, self.dtype),
                   np.empty(self.shape, self.dtype), np.empty(self.shape, self.dtype))
        shapes = (self.shape, (3,) + self.shape, self.shape, self.shape)
        ptrs = []
        for a, shape, name in zip(out, shapes, ("phi", "u", "p", "T")):
            ptr, _ = _host_ptr(a, self.dtype, shape, name, output=True)
            ptrs.append(C.c_void_p(ptr) if ptr is not None else None)
        _check(self._L.lbm_read_macro(self._h, *ptrs), "lbm_read_macro")
        return out

    def read_pops(self, which: int, stage: int = STAGE_STREAMED):
        out = np.empty((self.Q[which],) + self.shape, self.dtype)
        _check(self._L.lbm_read_pops(self._h, int(which), int(stage), C.c_void_p(out.ctypes.data)), "lbm_read_pops")
        return out

    def read_pops_noalloc(self, which: int, stage: int = STAGE_STREAMED):
        """read_pops without any device allocation (static scratch of NOALLOC_SCRATCH_BYTES; include/lbm.h)."""
        out = np.empty((self.Q[which],) + self.shape, self.dtype)
        _check(self._L.lbm_read_pops_noalloc(self._h, int(which), int(stage), C.c_void_p(out.ctypes.data)), "lbm_read_pops_noalloc")
        return out

    def save_state(self) -> np.ndarray:
        """lbm_save_state: the whole state as a byte array (header + workspace image) for lbm_load_state."""
        buf = np.empty(int(self._L.lbm_state_bytes(self._h)), dtype=np.uint8)
        _check(self._L.lbm_save_state(self._h, C.c_void_p(buf.ctypes.data)), "lbm_save_state")
        return buf

    def load_state(self, buf: np.ndarray):
        """lbm_load_state: continue from an image saved by a context of the same grid, lattice set and precision."""
        buf = np.ascontiguousarray(buf, dtype=np.uint8)
        if buf.size != int(self._L.lbm_state_bytes(self._h)):
            raise ValueError("state image of %d bytes, this context needs %d" % (buf.size, int(self._L.lbm_state_bytes(self._h))))
        _check(self._L.lbm_load_state(self._h, C.c_void_p(buf.ctypes.data)), "lbm_load_state")

    def note_replay(self, steps: int, launches: int):
        """lbm_note_replay: account for steps run (or only recorded) by a CUDA graph of the caller's."""
        _check(self._L.lbm_note_replay(self._h, int(steps), int(launches)), "lbm_note_replay")

    def check_finite(self) -> int:
        """lbm_check_finite: number of non-finite values in the current state (0 = the run is still in its stable range)."""
        n = C.c_longlong(-1)
        _check(self._L.lbm_check_finite(self._h, C.byref(n)), "lbm_check_finite")
        return int(n.value)

    def sync(self):
        _check(self._L.lbm_sync(self._h), "lbm_sync")

    @property
    def workspace_tensor(self):
        """The torch tensor that holds the workspace (what a neighbouring process maps through CUDA IPC)."""
        return self._ws

    @property
    def workspace_ptr(self) -> int:
        """Device address of the workspace lent to the library (what a neighbour maps for lbm_halo_push_mapped)."""
        return int(self._ws.data_ptr())

    @property
    def stream(self):
        """The torch.cuda.Stream every kernel and copy of this context is enqueued on (record timing events there)."""
        return self._stream

    def set_timing(self, enable: bool):
        _check(self._L.lbm_set_timing(self._h, 1 if enable else 0), "lbm_set_timing")

    def kernel_times(self):
        """(ms in K_phi, ms in K_main, timed steps) since the last call; synchronises."""
        a, b, n = C.c_double(), C.c_double(), C.c_longlong()
        _check(self._L.lbm_kernel_times(self._h, C.byref(a), C.byref(b), C.byref(n)), "lbm_kernel_times")
        return a.value, b.value, int(n.value)

    @property
    def step_count(self) -> int:
        return int(self._L.lbm_step_count(self._h))

    @property
    def launch_count(self) -> int:
        return int(self._L.lbm_launch_count(self._h))

    @property
    def variant(self) -> str:
        return self._L.lbm_variant(self._h).decode()

    def destroy(self):
        if getattr(self, "_h", None):
            self._L.lbm_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
