/*
 * lbm.h -- C ABI of the B200-native coupled phase-field lattice Boltzmann step.
 *
 * The library advances, per time step, the three coupled BGK lattice Boltzmann distributions of
 * Verdier, Kestener, Cartalade (arXiv 2003.06342; citations are PAPER.md:<line>):
 *   f  incompressible Navier-Stokes with surface tension, buoyancy and phase-change source
 *      (Eq.26a,b 27a-d 28a,b),
 *   g  conservative Allen-Cahn phase field, modified-equilibrium form (Eq.31a,b 32),
 *   s  temperature with latent-heat source (Eq.33a-d 34),
 * coupled through grad phi / lap phi (Eq.35,36), the chemical potential (Eq.14;
 * PAPER.md:118) and the production rate (Eq.18).  Every step of that path runs in
 * hand-written sm_100a CUDA kernels; there is no CPU fallback.  The readings taken where the paper is
 * garbled or silent are listed in DESIGN.md.
 *
 * Conventions
 *   - Fields are x-fastest, [z][y][x]; vector fields [comp][z][y][x] with 3 components (u_z = 0 in 2D);
 *     populations [Q][z][y][x] in the direction order documented in DESIGN.md ("Lattices").
 *   - "h_" pointers are HOST memory (pageable or pinned), "d_" pointers are DEVICE memory.
 *   - Element type of every field pointer is the context's precision: double (64) or float (32).
 *   - Precisions.  64: double storage and arithmetic (parity bar 1e-10 against the oracle).  32: float populations,
 *     production field, macro arrays and arithmetic -- except the phase-field path, which is kept wide because what its
 *     rounding adds to dphi/dt reaches T multiplied by L/Cp: the padded phi arrays are double,
 *     phi^{n+1} = sum_i g_i (Eq.32) is an exact sum of the float populations, dphi/dt = (phi^{n+1} - phi^n)/dt (Eq.34,
 *     DESIGN.md reading S4) and the collision of g (Eq.31) are evaluated in double.  Parity bar: 1e-4 relative to the
 *     oracle.  LBM_HALO_PHI buffers hold doubles in both precisions.
 *   - All calls return 0 (LBM_OK) or a negative LBM_E_* code; nothing throws across this boundary.
 *   - A context is bound to one device, one stream; calls on one context must not race.
 */
#ifndef LBM_H
#define LBM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* lattices, PAPER.md:190 (D2Q5 is not in the paper: DESIGN.md reading S1) */
enum { LBM_D2Q5 = 0, LBM_D2Q9 = 1, LBM_D3Q7 = 2, LBM_D3Q19 = 3, LBM_D3Q15 = 4 };

/* boundary rule of f on a face */
enum {
    LBM_F_PERIODIC = 0,
    LBM_F_WALL = 1, /* no-slip half bounce-back */
    LBM_F_OPEN = 2  /* pressure anti-bounce-back f_i = -f*_ibar + 2 w_i p_face (reading S12) */
};
/* boundary rule of g (phase field) and s (temperature) on a face */
enum {
    LBM_S_PERIODIC = 0,
    LBM_S_ZEROFLUX = 1, /* bounce-back */
    LBM_S_DIRICHLET = 2 /* anti-bounce-back s_i = -s*_ibar + 2 w_i value */
};

/* Model variants the paper defines beside the scheme it runs.  Both default to 0 = the paper's scheme;
 * a non-zero value runs the step on the plain direct kernel (parity-tested, not tuned) and stores u, p, T every step.
 * grad_scheme: directional derivative e_i.grad(phi) inside the gradient Eq.(35b): central Eq.(35a), or the biased differences
 *   of PAPER.md:318, first order [phi(x+e) - phi(x)]/dx (assembled over all directions it equals the central gradient up to
 *   rounding) and second order [-phi(x+2e) + 4 phi(x+e) - 3 phi(x)]/(2 dx).  The Laplacian stays Eq.(36).
 * div_scheme: div(u phi) of Eq.(33d),(34): product rule u.grad(phi) + phi mdot (1/rho_g - 1/rho_l), mdot the mass production rate
 *   (reading S5), or Eq.(35a,b) applied to the components of u phi with u and phi of the same level (reading S17:
 *   one more pass per step for the velocity; ghost velocity odd in no-slip walls, even in open faces).
 * Not available on slab contexts (halo) -- the ghost layers are one deep. */
enum { LBM_GRAD_CENTRAL = 0, LBM_GRAD_BIASED1 = 1, LBM_GRAD_BIASED2 = 2 };
enum { LBM_DIV_PRODUCT = 0, LBM_DIV_STENCIL = 1 };

/* flags */
#define LBM_FLAG_PHASE_CHANGE 1u /* production rate Eq.(18) on (otherwise m''' = 0)        */
#define LBM_FLAG_LATENT_HEAT 2u  /* source of the heat equation Eq.(33c,d),(34) on          */
#define LBM_FLAG_PRESCRIBED_U 4u /* u stays the field given to lbm_init (Zalesak / vortex verifications); */
                                 /* f is still stepped (its p is reported) but its first moment is ignored             */
/* Kernel selection.  The defaults are chosen by measurement per precision and grid; these flags force
 * the plainer kernels (all are parity-tested; results agree to rounding).  They change speed, never the method. */
#define LBM_FLAG_POPS_GATHER 16u  /* K_main gathers the populations into registers                                         */
#define LBM_FLAG_POPS_STAGED 32u  /* K_main stages the populations in shared memory with cp.async (the default, except for    */
                                  /* fp32 3D grids that cannot pair: odd or narrow rows, LBM_FLAG_ONE_NODE)                */
#define LBM_FLAG_PHI_LDG 64u      /* K_main reads the phi stencil through L1 instead of a TMA box                         */
#define LBM_FLAG_NO_PDL 256u      /* K_main not launched with programmatic dependent launch behind K_phi                  */
#define LBM_FLAG_ONE_NODE 512u    /* fp32 3D: K_main with one node per thread instead of a pair of x-adjacent nodes           */
#define LBM_FLAG_NO_GRAPH 128u    /* no CUDA-graph replay of the steps of small grids                                      */

/* error codes */
enum {
    LBM_OK = 0,
    LBM_E_INVALID = -1,   /* bad argument / parameter combination                         */
    LBM_E_UNSUPPORTED = -2, /* lattice set or precision not built                          */
    LBM_E_WORKSPACE = -3, /* workspace too small or misaligned                             */
    LBM_E_CUDA = -4,      /* a CUDA runtime call failed (lbm_last_cuda_error for the code) */
    LBM_E_STATE = -5,     /* call not valid in this state (e.g. step before init)          */
    LBM_E_NODEVICE = -6,  /* no sm_100 device / kernels not loadable                       */
    LBM_E_TOOLARGE = -7   /* lbm_read_pops_noalloc: the lattice does not fit the static scratch array */
};

/* which-population selectors and stages of lbm_read_pops */
enum { LBM_POPS_F = 0, LBM_POPS_G = 1, LBM_POPS_S = 2 };
enum {
    LBM_STAGE_POSTCOLLISION = 0, /* what the library stores: collided at the current level, not streamed */
    LBM_STAGE_STREAMED = 1       /* arrived at the node at the current level (post-pull, post-BC);        */
                                 /* needs at least one step since init                                   */
};

/*
 * Problem description; plain data, copied by lbm_create.
 * nz == 1 selects 2D (lattices must be D2Q*), nz > 1 selects 3D (D3Q*).
 * Supported lattice sets (f, g, s): (D2Q9, D2Q9, D2Q5), (D2Q9, D2Q9, D2Q9), (D3Q19, D3Q7, D3Q7), (D3Q15, D3Q7, D3Q7).
 * bc_*[axis][side]: axis 0,1,2 = x,y,z; side 0 = low face, 1 = high face.  A periodic face must be
 * periodic on both sides and for all three distributions (except next to a ghost layer, see halo).
 * Walls sit half a cell outside the first/last node (node i is at (i + 1/2) dx).
 *
 * halo[side] (slab decomposition of the paper's multi-GPU runs): the context holds one slab of a
 * larger domain cut along the SLOWEST axis (z in 3D, y in 2D).  halo[0] = 1 declares the first layer of that axis,
 * halo[1] = 1 the last one, a GHOST layer: a copy of the neighbouring slab's boundary layer, refreshed by the
 * caller with lbm_halo_pack / lbm_halo_unpack between the two phases of a step (lbm_step_phase).  nz (ny in 2D)
 * COUNTS the ghost layers; the three face kinds on a ghost side must be PERIODIC (the ghost layer is updated like any
 * node and its results are discarded), while the other side of the axis keeps its own kind.  Arrays given to
 * lbm_init and returned by lbm_read_* include the ghost layers; lbm_init wants valid phi, T, u, p there.
 */
typedef struct lbm_params {
    int nx, ny, nz;
    int lat_f, lat_g, lat_s;
    int precision;          /* 64 or 32 (see "Precisions" above)                                   */
    int bc_f[3][2];         /* LBM_F_*                                                              */
    int bc_g[3][2];         /* LBM_S_* for the phase field                                          */
    int bc_s[3][2];         /* LBM_S_* for the temperature                                          */
    double bc_phi[3][2];    /* Dirichlet value of phi per face                                      */
    double bc_T[3][2];      /* Dirichlet value of T per face                                        */
    double bc_p[3][2];      /* pressure of LBM_F_OPEN faces                                         */
    double dx, dt;          /* space and time step; c = dx/dt                                       */
    double rho_l, rho_g;    /* bulk densities, Eq.(1a)                                              */
    double nu_l, nu_g;      /* kinematic viscosities, harmonic interpolation Eq.(1b)                */
    double sigma, W, M;     /* surface tension, interface width, mobility (Eq.15b, 5)               */
    double grav[3];         /* gravity acceleration g; F_v = (rho - rho_l) g (reading G6) */
    double force[3];        /* uniform body force density added to F_tot             */
    double alpha_l, alpha_g;/* thermal diffusivities, linear in phi (reading S6)          */
    double L_latent, Cp;    /* latent heat and specific heat; theta = Cp (T - T_sat)/L              */
    double T_sat, theta_I;  /* saturation temperature; dimensionless interface temperature          */
    double A;               /* script-A of Eq.(18): 10/48 in the paper               */
    double eps_n;           /* n = grad phi / sqrt(|grad phi|^2 + eps_n^2) (reading S7)   */
    unsigned flags;         /* LBM_FLAG_*                                                           */
    int halo[2];            /* ghost layer on the low / high side of the slowest axis (0 or 1)      */
    int grad_scheme;        /* LBM_GRAD_*                                              */
    int div_scheme;         /* LBM_DIV_*                                                             */
} lbm_params;

typedef struct lbm_ctx lbm_ctx;

/* Bytes of device memory a context for *p needs (0 if p is invalid).  The caller allocates it (e.g. with
 * torch.empty(..., device="cuda")), 256-byte aligned, and lends it to the context until lbm_destroy. */
size_t lbm_workspace_bytes(const lbm_params *p);

/* Validate *p and build a context on the current CUDA device.  d_workspace: DEVICE pointer, >= bytes from
 * lbm_workspace_bytes, borrowed (never freed by the library).  cuda_stream: a cudaStream_t (NULL = legacy
 * default stream) on which every kernel and copy of this context is enqueued.  *out receives the context
 * (owned by the library; release with lbm_destroy). */
int lbm_create(const lbm_params *p, void *d_workspace, size_t bytes, void *cuda_stream, lbm_ctx **out);

/* Pointer arguments named h_* below are HOST pointers or, equally, DEVICE pointers of the context's device: the copies use
 * unified addressing (cudaMemcpyDefault), so a caller that keeps its fields on the GPU passes them directly.
 *
 * Set the state of time level 0 from HOST arrays (element type = precision).  h_phi is required; h_T, h_u,
 * h_p may be NULL (T = T_sat, u = 0, p = 0).  Sets dphi/dt = 0, the production field from the initial macros
 * (Eq.18) and the populations to bar-equilibrium theta_eq - dt/2 S (Eq.24; DESIGN.md reading
 * S9), then collides once so that the stored state is post-collision at level 0.  Resets the step counter.
 * Synchronises the stream before returning (the host arrays may be reused at once). */
int lbm_init(lbm_ctx *c, const void *h_phi, const void *h_T, const void *h_u, const void *h_p);

/* Enqueue n full coupled steps (each: K_phi = pull g + Eq.32, then K_main = stencils, closures, moments,
 * production refresh, collision of f, g, s) on the context's stream.  Asynchronous: returns after the
 * launches; launch errors are returned, execution errors surface at the next synchronising call.
 * The last of the n steps also stores u, p, T for lbm_read_macro. */
int lbm_step(lbm_ctx *c, int n);

/* LBM_FLAG_PRESCRIBED_U only: replace the prescribed velocity by the HOST array h_u ([3][nz][ny][nx], element type
 * = precision; the third component is ignored in 2D).  The field is u of the NEXT time level: the next step takes its
 * moments (T, p) and collides with it (time-dependent velocity of the reversing vortex).
 * Synchronises the stream.  LBM_E_INVALID without the flag, LBM_E_STATE before lbm_init. */
int lbm_set_velocity(lbm_ctx *c, const void *h_u);

/* ---- slab decomposition (contexts with halo[0] | halo[1]; lbm_step itself returns LBM_E_STATE for them) ----------
 * One step of a slab is   lbm_step_phase(c, 0, .)  -> exchange LBM_HALO_PHI ->  lbm_step_phase(c, 1, macros)
 * -> exchange LBM_HALO_POPS.   After lbm_init one LBM_HALO_POPS exchange is due before the first step.
 * phase 0 = K_phi (phi^{n+1} of every layer, Eq.32); phase 1 = K_main (moments, production, collisions) and the
 * buffer flip; store_macros != 0 also stores u, p, T.  Both are asynchronous on the context's stream.
 *
 * An exchange of `what` towards `side`: the sender packs its boundary layer next to its ghost side with
 * lbm_halo_pack(c, what, side, d_buf) into a DEVICE buffer of lbm_halo_bytes(c, what) bytes, the buffer travels to the
 * neighbour on that side (NCCL send/recv, a peer copy, or the same buffer when both slabs live in one process), and the
 * neighbour unpacks it into its ghost layer of the OPPOSITE side with lbm_halo_unpack(c, what, 1 - side, d_buf).
 *   LBM_HALO_PHI : the padded phi^{n+1} layer (with its in-layer ghost images);
 *   LBM_HALO_POPS: the post-collision populations that stream across the cut, i.e. those with e_axis = +1 for
 *                  side 1 and e_axis = -1 for side 0 (5 + 1 + 1 of D3Q19/D3Q7/D3Q7; 3 + 3 + 1 or 3 in 2D), whole layers.
 * pack / unpack are one kernel launch each, asynchronous on the context's stream; the caller orders the transfer
 * after the pack and the unpack after the transfer.  LBM_E_INVALID if the context has no ghost layer on that side. */
enum { LBM_HALO_PHI = 0, LBM_HALO_POPS = 1 };
int lbm_step_phase(lbm_ctx *c, int phase, int store_macros);

/* A phase in parts, for schedules that overlap the exchange with the interior (boundary layers first; PAPER.md:324, 559 is
 * the paper's decomposition, the overlap is this library's): run `phase` on the layers [first, first + count) of the slowest
 * axis only.  The caller covers every layer whose results it needs exactly once per phase -- the ghost layers need none: what
 * a step reads from them arrives by lbm_halo_unpack -- and marks the last part with last != 0, which completes the phase
 * (after phase 1 the buffers flip).  count == 0 is allowed (a bare "last").  While parts of phase 0 are outstanding
 * LBM_HALO_PHI may already be packed (from layers done) and unpacked; while parts of phase 1 are outstanding LBM_HALO_POPS
 * refers to the populations being written by this step.  Ordering between the parts, the packs and the transfers on the
 * device is the caller's (one stream, or events between two: lbm_set_stream).  Not with LBM_FLAG_PRESCRIBED_U unless the
 * one part is the whole grid. */
int lbm_step_layers(lbm_ctx *c, int phase, int first, int count, int store_macros, int last);

/* Enqueue the following calls of this context on another cudaStream_t (e.g. the packs and unpacks on an exchange stream while
 * the interior runs on the compute stream).  The caller orders the streams with events. */
int lbm_set_stream(lbm_ctx *c, void *cuda_stream);
int lbm_halo_bytes(const lbm_ctx *c, int what, size_t *bytes);
int lbm_halo_pack(lbm_ctx *c, int what, int side, void *d_buf);
int lbm_halo_unpack(lbm_ctx *c, int what, int side, const void *d_buf);
/* Pack and unpack in one launch where the neighbour's workspace can be addressed from this device (the same GPU, or a peer-mapped
 * workspace over NVLink): the boundary layer next to the ghost side `side` of c goes straight into the ghost layer of the OPPOSITE
 * side of `peer`, with no buffer in between.  Both contexts must stand at the same point of the same step (LBM_E_STATE otherwise)
 * and describe slabs of one domain (same lattice set, precision, nx, ny).  Enqueued on c's stream; the caller orders it against the
 * kernels of `peer` that read the ghost layer. */
int lbm_halo_push(lbm_ctx *c, int what, int side, lbm_ctx *peer);
/* The same for a neighbour that lives in ANOTHER process or on another GPU: *peer_params are the parameters its context was created
 * with and d_peer_workspace is its workspace as mapped into this process (CUDA IPC / peer access: a device pointer valid on the
 * current device).  The neighbour is taken to stand where c stands -- the slabs of a domain step in lockstep; ordering across the
 * processes (inter-process events) is the caller's. */
int lbm_halo_push_mapped(lbm_ctx *c, int what, int side, const lbm_params *peer_params, void *d_peer_workspace);
/* Ordering between processes without the host: lbm_stream_signal enqueues, on the context's stream, the write of `value` to the
 * 32-bit word d_flag (typically in the neighbour's peer-mapped memory) once everything enqueued before it -- the pushes -- is
 * visible; lbm_stream_wait holds the context's stream until the word d_flag (in this process's memory) is >= value (as a wrapping
 * signed difference).  Both are stream memory operations of the driver: no kernel spins and no host call blocks.
 * LBM_E_UNSUPPORTED where the driver does not offer them. */
int lbm_stream_signal(lbm_ctx *c, void *d_flag, unsigned value);
int lbm_stream_wait(lbm_ctx *c, void *d_flag, unsigned value);

/* Copy the macroscopic fields of the current time level to HOST arrays; any pointer may be NULL.
 * h_u is [3][z][y][x].  Synchronises. */
int lbm_read_macro(lbm_ctx *c, void *h_phi, void *h_u, void *h_p, void *h_T);

/* Debug / parity access: copy populations [Q][z][y][x] of lattice `which` at `stage` to HOST.  Synchronises.
 * Not on the hot path. */
int lbm_read_pops(lbm_ctx *c, int which, int stage, void *h_pops);

/* lbm_read_pops for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc).  lbm_read_pops stages the streamed populations (LBM_STAGE_STREAMED: the pull of PAPER.md:175 with the
 * boundary rules of PAPER.md:285, 418 applied) in a temporary from cudaMalloc; this call stages them in a file-scope
 * static __device__ array of LBM_NOALLOC_SCRATCH_BYTES bytes instead and calls no cudaMalloc, cudaFree or allocating
 * library routine.  Same arguments, same result.  Limits and sharing:
 *   - Q * nx * ny * nz * sizeof(element) of lattice `which` must be <= LBM_NOALLOC_SCRATCH_BYTES, else LBM_E_TOOLARGE
 *     (e.g. D3Q19 in double: 55 188 nodes, 38^3; D2Q9 in double: 116 508 nodes, 341^2);
 *   - every GPU that loads the library holds the array until the process exits;
 *   - ALL contexts of a device share the one array, which keeps the last call's contents.  The call overwrites the part it
 *     reads back (nothing has to start at zero) and returns after its own copy has finished, but two calls that overlap on
 *     the GPU (different contexts on different streams or host threads) race: serialise them;
 *   - the context's device must be current (as for every call); the array's device address is resolved once per device. */
#define LBM_NOALLOC_SCRATCH_BYTES (8u << 20)
int lbm_read_pops_noalloc(lbm_ctx *c, int which, int stage, void *h_pops);

/* Block until everything enqueued on the context's stream has finished; returns LBM_E_CUDA on a fault. */
int lbm_sync(lbm_ctx *c);

/* Checkpoint / resume.  lbm_save_state copies the whole state of the context (a 64-byte header and the workspace image:
 * lbm_state_bytes bytes) to the HOST buffer h_state; lbm_load_state puts such an image back into a context created for the same
 * grid, lattice set and precision (else LBM_E_INVALID; the physical parameters are the caller's business) -- also one that was never
 * initialised.  The restored context continues bit for bit.  Between steps only (LBM_E_STATE inside a phased step); both synchronise. */
size_t lbm_state_bytes(const lbm_ctx *c);
int lbm_save_state(lbm_ctx *c, void *h_state);
int lbm_load_state(lbm_ctx *c, const void *h_state);

/* Number of values of the current state (post-collision populations, production field, phi) that are not finite -> *n_bad.
 * The explicit scheme can leave its stable range (low mobility) and lbm_step never looks; this call does, off the
 * hot path (one pass over the state, no allocation: it uses the context's scratch field; synchronises). */
int lbm_check_finite(lbm_ctx *c, long long *n_bad);

/* Per-kernel device timing for measurement (off by default).  While enabled, lbm_step brackets K_phi and K_main of
 * every step (at most 4096 steps between two lbm_kernel_times calls) with CUDA events on the context's stream.
 * lbm_kernel_times synchronises, returns the summed durations in milliseconds and the number of timed steps,
 * and clears the record.  Any output pointer may be NULL. */
int lbm_set_timing(lbm_ctx *c, int enable);
int lbm_kernel_times(lbm_ctx *c, double *ms_phi, double *ms_main, long long *steps);

/* Counters: steps taken since init; kernels launched by this context since creation. */
/* For callers that capture lbm_step_layers / lbm_halo_* calls in a CUDA graph of their own (slabs.py does for small slabs): the
 * calls made during capture only record, and a replay runs them without the library seeing it -- add `steps` and `launches`
 * (either may be negative) to the context's counters.  The buffer parity is the caller's to keep: capture an even number of steps. */
int lbm_note_replay(lbm_ctx *c, long long steps, long long launches);
long long lbm_step_count(const lbm_ctx *c);
long long lbm_launch_count(const lbm_ctx *c);

/* Name of the kernel variant the context steps with, for logs: "gather+smem", "gather+phi-tma", "direct" (one node per thread:
 * populations staged in shared memory / gathered into registers with the phi tile by TMA / everything through L1), "pair+smem",
 * "pair+phi-tma" (fp32 3D: two nodes per thread, staged / gathered), "direct (model variant)" (grad_scheme / div_scheme). */
const char *lbm_variant(const lbm_ctx *c);

/* Last CUDA runtime error code seen by this library (cudaError_t as int), 0 if none. */
int lbm_last_cuda_error(void);

const char *lbm_strerror(int code);

/* Release the host context (NULL-safe).  Does not free the borrowed workspace. */
void lbm_destroy(lbm_ctx *c);

#ifdef __cplusplus
}
#endif
#endif /* LBM_H */
