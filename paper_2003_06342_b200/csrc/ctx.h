// Host-side declarations shared by the C-ABI translation unit (lbm.cu) and the per-lattice-set instantiation units
// (inst_*.cu).  Not part of the public boundary (that is include/lbm.h).
#pragma once

#include "../../include/lbm.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <vector>

#include "kernels.cuh"
#include "pairs.cuh"

namespace lbm {

extern int g_last_cuda_error;

#define CK(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) { lbm::g_last_cuda_error = (int)e_; return LBM_E_CUDA; } \
    } while (0)

enum LatSet { SET_NONE = 0, SET_2D_995, SET_2D_999, SET_3D_1977, SET_3D_1577 };

struct Layout {
    long long N;
    int es, es_phi;   // bytes per element: populations / Pdot / macros / caller's arrays; padded phi arrays
    int ppx, ppy, ppz, pz, xpad;
    size_t phi_pad_elems;
    size_t off_f[2], off_g[2], off_s[2], off_phi[2], off_pdot[2], off_u, off_p, off_T, off_scratch, total;
};

// One implementation = one (lattice set, precision, tile shape); chosen once in lbm_create.
struct ImplOps {
    int (*init)(lbm_ctx *, const void *, const void *, const void *, const void *);
    int (*step)(lbm_ctx *, int);
    int (*step_phase)(lbm_ctx *, int, int);
    int (*step_layers)(lbm_ctx *, int, int, int, int, int);   // phase, first layer, count, store macros, last part of the phase
    int (*read_macro)(lbm_ctx *, void *, void *, void *, void *);
    int (*read_pops)(lbm_ctx *, int, int, void *);
    int (*read_pops_scratch)(lbm_ctx *, int, int, void *, void *, size_t);   // staged in a caller-given device scratch (noalloc.cu)
    int bx, by, bz;   // tile of nodes per CTA
};

// lbm.cu: validation, lattice set and workspace layout of a parameter block (also of a PEER's, lbm_halo_push_mapped)
int describe_params(const lbm_params *p, LatSet *set, Layout *L);

// defined in inst_*.cu (compiled in parallel); nx selects the tile shape
const ImplOps *ops_2d995_f64(int nx);
const ImplOps *ops_3d15_f64(int nx);
const ImplOps *ops_3d15_f32(int nx);
const ImplOps *ops_2d995_f32(int nx);
const ImplOps *ops_2d999_f64(int nx);
const ImplOps *ops_2d999_f32(int nx);
const ImplOps *ops_3d_f64(int nx);
const ImplOps *ops_3d_f32(int nx);

}  // namespace lbm

struct lbm_ctx {
    lbm_params P;
    lbm::Layout L;
    lbm::LatSet set;
    const lbm::ImplOps *ops;
    char *ws;
    cudaStream_t stream;
    int cur;       // buffer holding the post-collision populations of the current level
    int curphi;    // padded phi buffer of the current level
    bool inited;
    int phase;     // slab contexts: the phase lbm_step_phase expects next (0 or 1)
    bool partial;  // lbm_step_layers has run parts of that phase, its last part is still due
    long long nsteps, launches;
    lbm::DevParams<double> pd;
    lbm::DevParams<float> pf;
    lbm::DevParams<lbm::f2> pf2;   // pf with every value doubled into a pair (k_main_pair.cuh)
    int num_sms;
    // K_main variants: phi halo tile staged by TMA, one box per CTA (k_main_phitma.cuh) ...
    bool phi_tma;
    // ... and the pulled populations, phi^n, Pdot staged by per-thread cp.async (k_main_smem.cuh)
    bool pops_smem;
    bool pdl;   // K_main launched with programmatic stream serialisation behind K_phi
    bool pair;  // fp32 3D: K_main carries two x-adjacent nodes per thread (k_main_pair.cuh) ...
    bool pair_smem;   // ... with the pair's populations staged in shared memory (k_main_pair_smem) or gathered into registers
    int attr_done[12];   // kernel attributes set on this context's device: [MODE] K_main, [8 + MODE] the pair kernel
    // CUDA graph of two consecutive plain steps, for launch-bound (small) grids
    bool graph_ok;
    cudaGraphExec_t graph2;
    int graph_launches;
    CUtensorMap map_phi_tile[2];
    // optional per-kernel timing (lbm_set_timing): 3 events per step: before k_phi, between, after k_main
    bool timing;
    std::vector<cudaEvent_t> ev;
};
