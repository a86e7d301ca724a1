// Host side of the C ABI declared in include/lbm.h: parameter validation, workspace carving, launch loop.
// No torch types, no CPU fallback: every step of the path runs in the kernels of k_phi.cuh / k_main.cuh.
#include "../../include/lbm.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include <cudaTypedefs.h>

#include "ctx.h"

namespace lbm {
int g_last_cuda_error = 0;
}

namespace {

using namespace lbm;

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

int lattice_q(int id) {
    switch (id) { case LBM_D2Q5: return 5; case LBM_D2Q9: return 9; case LBM_D3Q7: return 7; case LBM_D3Q19: return 19; case LBM_D3Q15: return 15; }
    return 0;
}
bool lattice_3d(int id) { return id == LBM_D3Q7 || id == LBM_D3Q19 || id == LBM_D3Q15; }

LatSet lattice_set(const lbm_params *p) {
    if (p->lat_f == LBM_D2Q9 && p->lat_g == LBM_D2Q9 && p->lat_s == LBM_D2Q5) return SET_2D_995;
    if (p->lat_f == LBM_D2Q9 && p->lat_g == LBM_D2Q9 && p->lat_s == LBM_D2Q9) return SET_2D_999;
    if (p->lat_f == LBM_D3Q19 && p->lat_g == LBM_D3Q7 && p->lat_s == LBM_D3Q7) return SET_3D_1977;
    if (p->lat_f == LBM_D3Q15 && p->lat_g == LBM_D3Q7 && p->lat_s == LBM_D3Q7) return SET_3D_1577;
    return SET_NONE;
}

int validate(const lbm_params *p) {
    if (!p) return LBM_E_INVALID;
    if (p->nx < 2 || p->ny < 2 || p->nz < 1) return LBM_E_INVALID;
    if (p->precision != 64 && p->precision != 32) return LBM_E_INVALID;
    if (!lattice_q(p->lat_f) || !lattice_q(p->lat_g) || !lattice_q(p->lat_s)) return LBM_E_INVALID;
    const bool three_d = p->nz > 1;
    if (lattice_3d(p->lat_f) != three_d || lattice_3d(p->lat_g) != three_d || lattice_3d(p->lat_s) != three_d)
        return LBM_E_INVALID;
    if (lattice_set(p) == SET_NONE) return LBM_E_UNSUPPORTED;
    if ((double)p->nx * p->ny * p->nz * 19.0 > 4294967295.0) return LBM_E_INVALID;   // 32-bit element offsets
    if (!(p->dx > 0) || !(p->dt > 0) || !(p->W > 0) || !(p->rho_l > 0) || !(p->rho_g > 0)) return LBM_E_INVALID;
    if (!(p->nu_l > 0) || !(p->nu_g > 0) || !(p->M > 0) || !(p->alpha_l > 0) || !(p->alpha_g > 0)) return LBM_E_INVALID;
    if (!(p->Cp > 0) || p->L_latent == 0.0 || !(p->A > 0) || !(p->eps_n > 0) || !(p->sigma >= 0)) return LBM_E_INVALID;
    for (int a = 0; a < 3; ++a) {
        for (int s = 0; s < 2; ++s) {
            if (p->bc_f[a][s] < 0 || p->bc_f[a][s] > 2 || p->bc_g[a][s] < 0 || p->bc_g[a][s] > 2 ||
                p->bc_s[a][s] < 0 || p->bc_s[a][s] > 2) return LBM_E_INVALID;
        }
        // a face is periodic for all three distributions or for none
        for (int s = 0; s < 2; ++s) {
            const bool per = p->bc_f[a][s] == LBM_F_PERIODIC;
            if ((p->bc_g[a][s] == LBM_S_PERIODIC) != per || (p->bc_s[a][s] == LBM_S_PERIODIC) != per) return LBM_E_INVALID;
        }
        // both faces of an axis are periodic together, unless a ghost layer of a slab sits on the periodic side
        const bool per0 = p->bc_f[a][0] == LBM_F_PERIODIC, per1 = p->bc_f[a][1] == LBM_F_PERIODIC;
        const int slab_axis = three_d ? 2 : 1;
        if (per0 != per1) {
            if (a != slab_axis) return LBM_E_INVALID;
            if (!(per0 ? p->halo[0] : p->halo[1])) return LBM_E_INVALID;
        }
    }
    {   // ghost layers: 0 or 1 per side, on a periodic-kind face, and at least one owned layer in between
        const int slab_axis = three_d ? 2 : 1;
        const int len = three_d ? p->nz : p->ny;
        for (int s = 0; s < 2; ++s) {
            if (p->halo[s] != 0 && p->halo[s] != 1) return LBM_E_INVALID;
            if (p->halo[s] && p->bc_f[slab_axis][s] != LBM_F_PERIODIC) return LBM_E_INVALID;
        }
        if (len - p->halo[0] - p->halo[1] < 1) return LBM_E_INVALID;
    }
    if (p->grad_scheme < LBM_GRAD_CENTRAL || p->grad_scheme > LBM_GRAD_BIASED2) return LBM_E_INVALID;
    if (p->div_scheme < LBM_DIV_PRODUCT || p->div_scheme > LBM_DIV_STENCIL) return LBM_E_INVALID;
    if ((p->grad_scheme || p->div_scheme) && (p->halo[0] | p->halo[1])) return LBM_E_UNSUPPORTED;   // ghost layers are one deep
    return LBM_OK;
}

Layout make_layout(const lbm_params *p) {
    Layout L{};
    const size_t es = p->precision == 64 ? 8 : 4;             // populations, Pdot, macros, scratch
    const size_t esp = 8;                                     // phi is kept in double in every precision (include/lbm.h)
    L.es = (int)es; L.es_phi = (int)esp;
    L.N = (long long)p->nx * p->ny * p->nz;
    const int mult = (int)(16 / esp);                         // TMA: row pitch and box starts are multiples of 16 bytes
    L.xpad = mult;                                            // node 0 sits 16 bytes into the padded row
    L.ppx = (p->nx + 2 * mult + mult - 1) / mult * mult;
    L.ppy = p->ny + 2;
    L.pz = p->nz > 1 ? 1 : 0;
    L.ppz = p->nz + 2 * L.pz;
    L.phi_pad_elems = (size_t)L.ppx * L.ppy * L.ppz;
    const size_t N = (size_t)L.N;
    size_t o = 0;
    auto take = [&](size_t elems, size_t esz) { size_t r = o; o = align_up(o + elems * esz); return r; };
    for (int b = 0; b < 2; ++b) L.off_f[b] = take(N * lattice_q(p->lat_f), es);
    for (int b = 0; b < 2; ++b) L.off_g[b] = take(N * lattice_q(p->lat_g), es);
    for (int b = 0; b < 2; ++b) L.off_s[b] = take(N * lattice_q(p->lat_s), es);
    for (int b = 0; b < 2; ++b) L.off_phi[b] = take(L.phi_pad_elems, esp);
    for (int b = 0; b < 2; ++b) L.off_pdot[b] = take(N, es);   // one per population buffer
    L.off_u = take(3 * N, es);
    L.off_p = take(N, es);
    L.off_T = take(N, es);
    L.off_scratch = take(N, es);
    L.total = o;
    return L;
}

template <class real> DevParams<real> make_dev_params(const lbm_params *p, const Layout &L) {
    DevParams<real> d{};
    d.nx = p->nx; d.ny = p->ny; d.nz = p->nz; d.N = L.N;
    d.s0 = 0; d.s1 = p->nz > 1 ? p->nz : p->ny;   // K_phi / K_main launches cover every layer unless lbm_step_layers narrows them
    d.ppx = L.ppx; d.ppy = L.ppy; d.pz = L.pz; d.xpad = L.xpad; d.pplane = (long long)L.ppx * L.ppy;
    for (int a = 0; a < 3; ++a) {
        for (int s = 0; s < 2; ++s) {
            d.bc_f[a][s] = p->bc_f[a][s];   // PERIODIC 0, WALL -> BOUNCE 1, OPEN -> ANTI 2 (same numbering)
            d.bc_g[a][s] = p->bc_g[a][s];
            d.bc_s[a][s] = p->bc_s[a][s];
            d.bc_phi[a][s] = (real)p->bc_phi[a][s];
            d.bc_T[a][s] = (real)p->bc_T[a][s];
            d.bc_p[a][s] = (real)p->bc_p[a][s];
        }
        d.nonper[a] = p->bc_f[a][0] != LBM_F_PERIODIC || p->bc_f[a][1] != LBM_F_PERIODIC;   // one side may be a slab ghost side
        d.grav[a] = (real)p->grav[a];
        d.force[a] = (real)p->force[a];
    }
    if (p->nz == 1) d.nonper[2] = 0;
    d.bcfaces = 0;
    for (int a = 0; a < (p->nz == 1 ? 2 : 3); ++a)
        for (int s = 0; s < 2; ++s)
            if (p->bc_f[a][s] != LBM_F_PERIODIC) d.bcfaces |= 1u << (2 * a + s);
    const double c = p->dx / p->dt;
    auto e2 = [](int id) { return id == LBM_D3Q7 ? 0.25 : 1.0 / 3.0; };
    const double cs2f = e2(p->lat_f) * c * c, cs2g = e2(p->lat_g) * c * c, cs2s = e2(p->lat_s) * c * c;
    d.dt = (real)p->dt; d.hdt = (real)(0.5 * p->dt); d.c = (real)c;
    d.inv_dx = (real)(1.0 / p->dx); d.inv_dx2 = (real)(1.0 / (p->dx * p->dx));
    d.cs2f = (real)cs2f; d.cs2g = (real)cs2g; d.cs2s = (real)cs2s;
    d.inv_cs2f = (real)(1.0 / cs2f); d.inv_cs2g = (real)(1.0 / cs2g); d.inv_cs2s = (real)(1.0 / cs2s);
    d.c_cs2f = (real)(c / cs2f); d.c_cs2g = (real)(c / cs2g); d.c_cs2s = (real)(c / cs2s);
    d.inv_dt = (real)(1.0 / p->dt);
    d.tauf_num = (real)(p->nu_l * p->nu_g / (cs2f * p->dt));
    d.taus_den = (real)(1.0 / (cs2s * p->dt));
    d.rho_l = (real)p->rho_l; d.rho_g = (real)p->rho_g; d.rho_diff = (real)(p->rho_g - p->rho_l);
    d.drho = (real)(1.0 / p->rho_g - 1.0 / p->rho_l);
    d.nu_l = (real)p->nu_l; d.nu_g = (real)p->nu_g; d.nu_prod = (real)(p->nu_l * p->nu_g);
    d.fourH = (real)(4.0 * 12.0 * p->sigma / p->W);            // H = 12 sigma / W, Eq.(15b)
    d.K = (real)(1.5 * p->W * p->sigma);                       // K = 3/2 W sigma, Eq.(15b)
    d.alpha_l = (real)p->alpha_l; d.alpha_diff = (real)(p->alpha_g - p->alpha_l);
    d.M = (real)p->M;
    d.om_g = (real)(1.0 / (p->M / (cs2g * p->dt) + 0.5));      // PAPER.md:236, Eq.(25)
    d.cac = (real)(p->M * (4.0 / p->W) * c / cs2g);            // Eq.(31b) counter term factor
    d.g_om = 1.0 / (p->M / (cs2g * p->dt) + 0.5); d.g_dt = p->dt; d.g_c_cs2 = c / cs2g; d.g_inv_cs2 = 1.0 / cs2g;
    d.g_cac = p->M * (4.0 / p->W) * c / cs2g;
    d.LCp = (real)(p->L_latent / p->Cp); d.CpL = (real)(p->Cp / p->L_latent);
    d.T_sat = (real)p->T_sat; d.theta_I = (real)p->theta_I;
    d.pc_coef = (real)(4.0 / (p->A * p->W * p->W));            // Eq.(18)
    d.eps_n2 = (real)(p->eps_n * p->eps_n);
    d.phase_change = (p->flags & LBM_FLAG_PHASE_CHANGE) ? 1 : 0;
    d.latent_heat = (p->flags & LBM_FLAG_LATENT_HEAT) ? 1 : 0;
    d.prescribed_u = (p->flags & LBM_FLAG_PRESCRIBED_U) ? 1 : 0;
    d.grad_scheme = p->grad_scheme; d.div_scheme = p->div_scheme;
    return d;
}

}  // namespace

namespace {

PFN_cuTensorMapEncodeTiled_v12000 get_encode_fn() {
    static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
    }
    return fn;
}

// box tensor map of the padded phi buffers for the gather kernel's halo tile (k_main_phitma.cuh)
bool build_phi_tile_maps(lbm_ctx *c) {
    auto fn = get_encode_fn();
    if (!fn) return false;
    const int es = c->L.es_phi;
    const int epb = 16 / es;
    const bool three_d = c->P.nz > 1;
    for (int b = 0; b < 2; ++b) {
        cuuint64_t gdim[3] = {(cuuint64_t)c->L.ppx, (cuuint64_t)c->L.ppy, (cuuint64_t)c->L.ppz};
        cuuint64_t gstr[2] = {(cuuint64_t)c->L.ppx * es, (cuuint64_t)c->L.ppx * c->L.ppy * es};
        cuuint32_t box[3] = {(cuuint32_t)(c->ops->bx + 2 * epb), (cuuint32_t)(c->ops->by + 2),
                             (cuuint32_t)(three_d ? c->ops->bz + 2 : 1)};
        cuuint32_t estr[3] = {1, 1, 1};
        if (box[0] > 256 || gstr[0] % 16 != 0) return false;
        CUresult r = fn(&c->map_phi_tile[b], es == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3,
                        c->ws + c->L.off_phi[b], gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return false;
    }
    return true;
}

// Order of the work items of the single-launch step (k_step.cuh): rows per mid-axis block and lead of K_phi over K_main in
// layer pairs; 0 / negative = the defaults chosen by measurement.
}  // namespace

namespace lbm {
int describe_params(const lbm_params *p, LatSet *set, Layout *L) {
    const int rc = validate(p);
    if (rc) return rc;
    *set = lattice_set(p);
    *L = make_layout(p);
    return LBM_OK;
}
}  // namespace lbm

// ------------------------------------------------------------------------------------------------ C ABI
extern "C" {

size_t lbm_workspace_bytes(const lbm_params *p) {
    if (validate(p) != LBM_OK) return 0;
    return make_layout(p).total;
}

int lbm_create(const lbm_params *p, void *d_workspace, size_t bytes, void *cuda_stream, lbm_ctx **out) {
    if (!out) return LBM_E_INVALID;
    *out = nullptr;
    int rc = validate(p);
    if (rc) return rc;
    Layout L = make_layout(p);
    if (!d_workspace || bytes < L.total || (reinterpret_cast<size_t>(d_workspace) % ALIGN) != 0) return LBM_E_WORKSPACE;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        g_last_cuda_error = (int)cudaGetLastError();
        return LBM_E_NODEVICE;
    }
    if (prop.major != 10) return LBM_E_NODEVICE;   // kernels are built for sm_100a only
    cudaPointerAttributes attr;
    CK(cudaPointerGetAttributes(&attr, d_workspace));
    if (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) return LBM_E_WORKSPACE;
    lbm_ctx *c = new (std::nothrow) lbm_ctx();
    if (!c) return LBM_E_INVALID;
    c->P = *p; c->L = L; c->set = lattice_set(p);
    {
        const bool d = p->precision == 64;
        switch (c->set) {
        case SET_2D_995: c->ops = d ? ops_2d995_f64(p->nx) : ops_2d995_f32(p->nx); break;
        case SET_2D_999: c->ops = d ? ops_2d999_f64(p->nx) : ops_2d999_f32(p->nx); break;
        case SET_3D_1977: c->ops = d ? ops_3d_f64(p->nx) : ops_3d_f32(p->nx); break;
        case SET_3D_1577: c->ops = d ? ops_3d15_f64(p->nx) : ops_3d15_f32(p->nx); break;
        default: delete c; return LBM_E_UNSUPPORTED;
        }
    }
    c->ws = static_cast<char *>(d_workspace);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    c->cur = 0; c->curphi = 0; c->phase = 0; c->partial = false; c->inited = false; c->nsteps = 0; c->launches = 0; c->timing = false;
    c->pd = make_dev_params<double>(p, L);
    c->pf = make_dev_params<float>(p, L);
    c->pf2 = make_dev_params<f2>(p, L);
    c->num_sms = prop.multiProcessorCount;
    {   // Kernel variants, chosen by measurement; lbm_params.flags can force the plainer ones.
        const unsigned fl = p->flags;
        // small (launch-bound) grids replay their steps from a CUDA graph; the legacy default stream cannot be captured
        c->graph_ok = c->stream != nullptr && L.N <= (1ll << 21) && !(fl & LBM_FLAG_NO_GRAPH);
        c->graph2 = nullptr; c->graph_launches = 0;
        for (int &a : c->attr_done) a = 0;
        c->pdl = !(fl & LBM_FLAG_NO_PDL);
        // phi halo tile of K_main: one TMA box per CTA into shared memory (default) or plain loads through L1
        c->phi_tma = !(fl & LBM_FLAG_PHI_LDG) && build_phi_tile_maps(c);
        // pulled populations of K_main: staged in shared memory by cp.async (k_main_smem.cuh) where that measured faster --
        // fp64 (+3..9% on every large grid) and fp32 in 2D (+8%); fp32 3D stays on the register gather (-1..5%)
        const bool smem_default = p->precision == 64 || p->nz == 1;
        c->pops_smem = c->phi_tma && ((fl & LBM_FLAG_POPS_STAGED) ? true : (fl & LBM_FLAG_POPS_GATHER) ? false : smem_default);
        // fp32 3D on 128- or 64-wide tiles with even rows: two x-adjacent nodes per thread, packed f32x2 arithmetic (k_main_pair.cuh)
        c->pair = c->phi_tma && p->precision == 32 && p->nz > 1 && c->ops->bx >= 64 && p->nx % 2 == 0 && !(fl & LBM_FLAG_ONE_NODE);
        c->pair_smem = c->pair && !(fl & LBM_FLAG_POPS_GATHER);
        if (c->pair) c->pops_smem = false;
    }
    *out = c;
    return LBM_OK;
}

int lbm_init(lbm_ctx *c, const void *h_phi, const void *h_T, const void *h_u, const void *h_p) {
    if (!c || !h_phi) return LBM_E_INVALID;
    return c->ops->init(c, h_phi, h_T, h_u, h_p);
}

int lbm_set_velocity(lbm_ctx *c, const void *h_u) {
    if (!c || !h_u || !(c->P.flags & LBM_FLAG_PRESCRIBED_U)) return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    const size_t es = (size_t)c->L.es;
    CK(cudaMemcpyAsync(c->ws + c->L.off_u, h_u, 3 * (size_t)c->L.N * es, cudaMemcpyDefault, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

int lbm_step(lbm_ctx *c, int n) {
    if (!c || n < 0) return LBM_E_INVALID;
    if (!c->inited || (c->P.halo[0] | c->P.halo[1])) return LBM_E_STATE;   // slabs step by phases (ghost exchange in between)
    if (c->phase != 0 || c->partial) return LBM_E_STATE;
    return c->ops->step(c, n);
}

int lbm_step_layers(lbm_ctx *c, int phase, int first, int count, int store_macros, int last) {
    if (!c || (phase != 0 && phase != 1)) return LBM_E_INVALID;
    const int nslow = c->P.nz > 1 ? c->P.nz : c->P.ny;
    if (first < 0 || count < 0 || first + count > nslow) return LBM_E_INVALID;
    if (!c->inited || phase != c->phase) return LBM_E_STATE;
    if ((c->P.flags & LBM_FLAG_PRESCRIBED_U) || c->P.grad_scheme || c->P.div_scheme) {
        if (first != 0 || count != nslow || !last) return LBM_E_UNSUPPORTED;
    }
    const int rc = c->ops->step_layers(c, phase, first, count, store_macros, last);
    if (rc) return rc;
    c->partial = !last;
    if (last) c->phase = 1 - phase;
    return LBM_OK;
}

int lbm_set_stream(lbm_ctx *c, void *cuda_stream) {
    if (!c) return LBM_E_INVALID;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    return LBM_OK;
}

int lbm_step_phase(lbm_ctx *c, int phase, int store_macros) {
    if (!c || (phase != 0 && phase != 1)) return LBM_E_INVALID;
    if (!c->inited || phase != c->phase || c->partial) return LBM_E_STATE;
    const int rc = c->ops->step_phase(c, phase, store_macros);
    if (rc == LBM_OK) c->phase = 1 - phase;
    return rc;
}

int lbm_read_macro(lbm_ctx *c, void *h_phi, void *h_u, void *h_p, void *h_T) {
    if (!c) return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    return c->ops->read_macro(c, h_phi, h_u, h_p, h_T);
}

int lbm_read_pops(lbm_ctx *c, int which, int stage, void *h_pops) {
    if (!c || !h_pops || which < 0 || which > 2 || (stage != LBM_STAGE_POSTCOLLISION && stage != LBM_STAGE_STREAMED))
        return LBM_E_INVALID;
    if (!c->inited) return LBM_E_STATE;
    return c->ops->read_pops(c, which, stage, h_pops);
}

int lbm_sync(lbm_ctx *c) {
    if (!c) return LBM_E_INVALID;
    CK(cudaStreamSynchronize(c->stream));
    return LBM_OK;
}

int lbm_set_timing(lbm_ctx *c, int enable) {
    if (!c) return LBM_E_INVALID;
    c->timing = enable != 0;
    return LBM_OK;
}

int lbm_kernel_times(lbm_ctx *c, double *ms_phi, double *ms_main, long long *steps) {
    if (!c) return LBM_E_INVALID;
    CK(cudaStreamSynchronize(c->stream));
    double a = 0.0, b = 0.0;
    const size_t n = c->ev.size() / 3;
    for (size_t k = 0; k < n; ++k) {
        float t0 = 0.f, t1 = 0.f;
        CK(cudaEventElapsedTime(&t0, c->ev[3 * k], c->ev[3 * k + 1]));
        CK(cudaEventElapsedTime(&t1, c->ev[3 * k + 1], c->ev[3 * k + 2]));
        a += t0; b += t1;
    }
    for (auto e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    if (ms_phi) *ms_phi = a;
    if (ms_main) *ms_main = b;
    if (steps) *steps = (long long)n;
    return LBM_OK;
}

int lbm_note_replay(lbm_ctx *c, long long steps, long long launches) {
    if (!c) return LBM_E_INVALID;
    if (c->nsteps + steps < 0 || c->launches + launches < 0) return LBM_E_INVALID;
    c->nsteps += steps; c->launches += launches;
    return LBM_OK;
}

long long lbm_step_count(const lbm_ctx *c) { return c ? c->nsteps : -1; }
long long lbm_launch_count(const lbm_ctx *c) { return c ? c->launches : -1; }
const char *lbm_variant(const lbm_ctx *c) {
    if (!c) return "";
    if (c->P.grad_scheme || c->P.div_scheme) return "direct (model variant)";
    if (c->pair) return c->pair_smem ? "pair+smem" : "pair+phi-tma";
    return c->phi_tma ? (c->pops_smem ? "gather+smem" : "gather+phi-tma") : "direct";
}
int lbm_last_cuda_error(void) { return g_last_cuda_error; }

const char *lbm_strerror(int code) {
    switch (code) {
    case LBM_OK: return "ok";
    case LBM_E_INVALID: return "invalid argument or parameter combination";
    case LBM_E_UNSUPPORTED: return "lattice set or precision not built";
    case LBM_E_WORKSPACE: return "workspace too small, misaligned or not device memory";
    case LBM_E_CUDA: return "CUDA runtime error (see lbm_last_cuda_error)";
    case LBM_E_STATE: return "call not valid in this state";
    case LBM_E_NODEVICE: return "no sm_100 CUDA device";
    case LBM_E_TOOLARGE: return "lattice larger than the static scratch array of the no-alloc entry point (LBM_NOALLOC_SCRATCH_BYTES)";
    default: return "unknown error";
    }
}

void lbm_destroy(lbm_ctx *c) {
    if (!c) return;
    for (auto e : c->ev) cudaEventDestroy(e);
    if (c->graph2) cudaGraphExecDestroy(c->graph2);
    delete c;
}

}  // extern "C"
