// Host-side implementation template: launches of one (lattice set, precision, tile shape).  Included by inst_*.cu only.
#pragma once

#include "ctx.h"
#include "k_main.cuh"
#include "k_main_pair.cuh"
#include "k_main_phitma.cuh"
#include "k_main_smem.cuh"
#include "k_phi.cuh"

namespace lbm {

// Tiles of nodes per CTA (one node per thread).  A warp is one x-row.  Wide tiles (long contiguous x-runs: fewer partially
// used sectors on the x-shifted pulls) are 3.5% faster on config 4 and are used when the row is long enough; narrow tiles
// keep small grids busy.  Wide tiles only when the ragged last tile wastes at most 4% of the threads (192 = 128 + 64
// would idle 25%; a 192-wide tile on nx = 192 measured 9% SLOWER than the narrow tile).
inline bool wide_tile_pays(int nx, int bx = 128) { return nx >= bx && ((nx + bx - 1) / bx * bx - nx) * 25 <= nx; }

// K_phi and the utility kernels always run 256-thread tiles (PhiTile).  K_main on wide tiles runs 128-thread CTAs, one
// x-row each (finer CTA turnover at the same number of warps: +3% fp64 3D, +7% fp64 2D, +7% fp32 2D), except in fp32 3D
// where 128 x 2 is faster (measured).
struct TileWide3Phi { static constexpr int BX = 128, BY = 2, BZ = 1; using PhiTile = TileWide3Phi; };   // fp32 3D K_main too
struct TileWide3 { static constexpr int BX = 128, BY = 1, BZ = 1; using PhiTile = TileWide3Phi; };
struct TileNarrow3 { static constexpr int BX = 32, BY = 4, BZ = 2; using PhiTile = TileNarrow3; };
struct TileMid3Phi { static constexpr int BX = 64, BY = 4, BZ = 1; using PhiTile = TileMid3Phi; };
// rows that are a multiple of 64 where the 128-wide tile does not pay (192, 320): 64 x 2 instead of the narrow tile, 3D:
// config 5 at 192^3 9759 -> 10 019 MLUPS (bench.py), 320^3 9856 -> 10 213 (probe); fp32 3D: 192^3 15 719 -> 16 853, 320^3 16 285 -> 17 386
struct TileMid3 { static constexpr int BX = 64, BY = 2, BZ = 1; using PhiTile = TileMid3Phi; };
struct TileWide2 { static constexpr int BX = 128, BY = 2, BZ = 1; using PhiTile = TileWide2; };
struct TileWide2K { static constexpr int BX = 128, BY = 1, BZ = 1; using PhiTile = TileWide2; };
struct TileNarrow2 { static constexpr int BX = 32, BY = 8, BZ = 1; using PhiTile = TileNarrow2; };

// grid of a K_phi / K_main launch over the layers [pd.s0, pd.s1) of the slowest axis (lbm_ctx::pd, pf carry the same range)
template <class T> dim3 grid_layers(const lbm_ctx *c) {
    const lbm_params &P = c->P;
    const int n = c->pd.s1 - c->pd.s0;
    if (P.nz > 1) return dim3((P.nx + T::BX - 1) / T::BX, (P.ny + T::BY - 1) / T::BY, (n + T::BZ - 1) / T::BZ);
    return dim3((P.nx + T::BX - 1) / T::BX, (n + T::BY - 1) / T::BY, 1);
}

// Shared-memory carve-out (percent of the 228 KB maximum) for `ctas` resident CTAs of `bytes` dynamic shared memory each (+1 KB
// that the driver reserves per CTA): the smallest configuration of sm_100 that holds them, requested from below so that the
// rounding of the percentage cannot tip it into the next larger one.  The rest of the 256 KB stays L1 -- the shifted pulls of
// neighbouring warps share sectors there (measured on config 4, fp64 K_main ms: 60 KB of L1: 2.89, 92 KB: 2.82, and 3.75 with
// the maximum carve-out).
inline int carveout_pct(int ctas, size_t bytes) {
    const size_t need = (size_t)ctas * (bytes + 1024);
    const size_t sizes[] = {0, 8, 16, 32, 64, 100, 132, 164, 196, 228};
    size_t pick = 228;
    for (size_t s : sizes) if (s * 1024 >= need) { pick = s; break; }
    return (int)(pick * 1024 * 100 / 233472);
}

template <class real> const DevParams<real> &dev_params(const lbm_ctx *c);
template <> inline const DevParams<double> &dev_params<double>(const lbm_ctx *c) { return c->pd; }
template <> inline const DevParams<float> &dev_params<float>(const lbm_ctx *c) { return c->pf; }

template <class real> real *wsp(const lbm_ctx *c, size_t off) { return reinterpret_cast<real *>(c->ws + off); }

template <class T> dim3 grid_for(const lbm_params &P) {
    return dim3((P.nx + T::BX - 1) / T::BX, (P.ny + T::BY - 1) / T::BY, (P.nz + T::BZ - 1) / T::BZ);
}

// real: arithmetic type; sreal: storage of populations, Pdot, macros (and the type of the caller's arrays); preal: phi arrays.
template <class LF, class LG, class LS, class real, class T, class sreal = real, class preal = real> struct Impl {
    static constexpr int D = LF::D;
    static constexpr bool UNIFORM = std::is_same<real, sreal>::value && std::is_same<real, preal>::value;
    using Fields = DevFieldsT<sreal, preal>;
    static constexpr int NT = T::BX * T::BY * T::BZ;
    using TP = typename T::PhiTile;                       // tile of K_phi and of the utility kernels
    static constexpr int NTP = TP::BX * TP::BY * TP::BZ;
    // Threads per SM the register allocation is bounded for (__launch_bounds__ minimum CTAs = threads / NT), measured:
    //   fp64 3D: 512 (128 registers, no spill on the interior path); more spills cost more than the warps bring
    //   fp64 2D, 128-thread CTAs: 640 (96 registers; K_main with staged populations on 4096x3072, D2Q5 heat lattice:
    //            512 / 640 / 768 / 896 / 1024 threads: 0.785 / 0.752 / 0.754 / 0.792 / 0.854 ms; three D2Q9: 640 best);
    //            256-thread tiles 768
    //   fp32   : 1024 (64 registers; +25% over 512 although a few values spill); 2D with staged populations on 4096x3072,
    //            768 / 1024 / 1280 / 1536 threads: 0.481 / 0.470 / 0.506 / 0.570 ms (three D2Q9: 0.541 / 0.533 / 0.604 / 0.778)
    static constexpr int THREADS64 = D == 3 ? 512 : (NT == 128 ? 640 : 768);
    static constexpr int THREADS32 = 1024;
    static constexpr int MINB = (sizeof(real) == 8 ? THREADS64 : THREADS32) / NT;
    static constexpr int PHI_NPT = 2;   // nodes per thread in K_phi (1: 0.427 ms, 2: 0.378, 4: 0.447 on config 4 fp64)
    static Fields fields(const lbm_ctx *c, int in, int out, int phi_new, int phi_old) {
        Fields F{};
        F.f_in = wsp<sreal>(c, c->L.off_f[in]);  F.f_out = wsp<sreal>(c, c->L.off_f[out]);
        F.g_in = wsp<sreal>(c, c->L.off_g[in]);  F.g_out = wsp<sreal>(c, c->L.off_g[out]);
        F.s_in = wsp<sreal>(c, c->L.off_s[in]);  F.s_out = wsp<sreal>(c, c->L.off_s[out]);
        F.phi_new = wsp<preal>(c, c->L.off_phi[phi_new]);
        F.phi_old = wsp<preal>(c, c->L.off_phi[phi_old]);
        // the production field lives with its population buffer: level n in [in], level n+1 into [out] (the rest population
        // of g in a buffer carries dt/2 Pdot of the SAME buffer, k_main.cuh)
        F.pdot_in = wsp<sreal>(c, c->L.off_pdot[in]);
        F.pdot = wsp<sreal>(c, c->L.off_pdot[out]);
        F.u = wsp<sreal>(c, c->L.off_u); F.p = wsp<sreal>(c, c->L.off_p); F.T = wsp<sreal>(c, c->L.off_T);
        return F;
    }

    // kernel attributes are per device: set once per context (lbm_create may run on any device of the process)
    template <class K> static int set_smem_attrs(lbm_ctx *c, K kern, size_t bytes, int &done_flag) {
        if (done_flag) return LBM_OK;
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carveout_pct(MINB, bytes)));
        done_flag = 1;
        return LBM_OK;
    }

    // K_main right behind K_phi in the stream, with programmatic dependent launch (unless LBM_FLAG_NO_PDL): its CTAs may start
    // while K_phi drains; they wait (griddepcontrol.wait, k_main_*.cuh) before they request their phi box
    template <class K> static cudaError_t launch_after_phi(lbm_ctx *c, K kern, size_t smem, const DevParams<real> &P, const Fields &F,
                                                           const CUtensorMap &map) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid_layers<T>(c); cfg.blockDim = dim3(NT); cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = c->pdl ? 1 : 0;
        return cudaLaunchKernelEx(&cfg, kern, P, F, map);
    }

    // two nodes per thread (k_main_pair.cuh): float populations with a double phi, 3D, 128- or 64-wide tiles, even rows
    static constexpr bool PAIRABLE = D == 3 && std::is_same<real, float>::value && std::is_same<sreal, float>::value &&
                                     std::is_same<preal, double>::value && (T::BX == 128 || T::BX == 64);
    static constexpr int PAIR_THREADS = 512;   // per SM: 128 registers per thread, as the double-precision kernel

    template <int MODE> static int launch_main(lbm_ctx *c, const Fields &F, int pnew = 0) {
        if constexpr (MODE == MODE_STEP || MODE == MODE_STEP_MACRO) {
            if constexpr (PAIRABLE) {
                if (c->pair) {
                    constexpr int PMINB = PAIR_THREADS / (NT / 2);
                    using PC = PairSmemCfg<LF, LG, LS, T::BX, T::BY, T::BZ>;
                    auto kern = c->pair_smem ? k_main_pair_smem<LF, LG, LS, MODE, T::BX, T::BY, T::BZ, PMINB, Fields>
                                             : k_main_pair<LF, LG, LS, MODE, T::BX, T::BY, T::BZ, PMINB, Fields>;
                    if (c->pair_smem && !c->attr_done[8 + MODE]) {   // per device: this context's first launch sets them
                        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PC::BYTES));
                        CK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, carveout_pct(PMINB, PC::BYTES)));
                        c->attr_done[8 + MODE] = 1;
                    }
                    cudaLaunchConfig_t cfg = {};
                    cfg.gridDim = grid_layers<T>(c); cfg.blockDim = dim3(NT / 2); cfg.stream = c->stream;
                    cfg.dynamicSmemBytes = c->pair_smem ? PC::BYTES : 0;
                    cudaLaunchAttribute at[1];
                    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                    at[0].val.programmaticStreamSerializationAllowed = 1;
                    cfg.attrs = at; cfg.numAttrs = c->pdl ? 1 : 0;
                    CK(cudaLaunchKernelEx(&cfg, kern, c->pf, c->pf2, F, c->map_phi_tile[pnew]));
                    c->launches++;
                    return LBM_OK;
                }
            }
            if (c->phi_tma && c->pops_smem) {
                using C = SmemCfg<LF, LG, LS, sreal, preal, T::BX, T::BY, T::BZ>;
                auto kern = k_main_smem<LF, LG, LS, real, MODE, T::BX, T::BY, T::BZ, MINB, Fields>;
                int rc = set_smem_attrs(c, kern, C::BYTES, c->attr_done[MODE]);
                if (rc) return rc;
                CK(launch_after_phi(c, kern, C::BYTES, dev_params<real>(c), F, c->map_phi_tile[pnew]));
                c->launches++;
                return LBM_OK;
            }
            if (c->phi_tma) {
                auto kern = k_main_phitma<LF, LG, LS, real, MODE, T::BX, T::BY, T::BZ, MINB, Fields>;
                CK(launch_after_phi(c, kern, 0, dev_params<real>(c), F, c->map_phi_tile[pnew]));
                c->launches++;
                return LBM_OK;
            }
        }
        k_main_direct<LF, LG, LS, real, MODE, T::BX, T::BY, T::BZ, MINB>
            <<<grid_layers<T>(c), NT, 0, c->stream>>>(dev_params<real>(c), F);
        c->launches++;
        CK(cudaGetLastError());
        return LBM_OK;
    }

    static int init(lbm_ctx *c, const void *h_phi, const void *h_T, const void *h_u, const void *h_p) {
        const size_t N = (size_t)c->L.N, es = sizeof(sreal);
        const DevParams<real> &P = dev_params<real>(c);
        sreal *scratch = wsp<sreal>(c, c->L.off_scratch);
        CK(cudaMemcpyAsync(scratch, h_phi, N * es, cudaMemcpyDefault, c->stream));
        sreal *dT = wsp<sreal>(c, c->L.off_T), *du = wsp<sreal>(c, c->L.off_u), *dp = wsp<sreal>(c, c->L.off_p);
        if (h_T) CK(cudaMemcpyAsync(dT, h_T, N * es, cudaMemcpyDefault, c->stream));
        else {
            k_fill<sreal><<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(dT, (long long)N, (sreal)c->P.T_sat);
            c->launches++;
            CK(cudaGetLastError());
        }
        if (h_u) CK(cudaMemcpyAsync(du, h_u, 3 * N * es, cudaMemcpyDefault, c->stream));
        else CK(cudaMemsetAsync(du, 0, 3 * N * es, c->stream));
        if (h_p) CK(cudaMemcpyAsync(dp, h_p, N * es, cudaMemcpyDefault, c->stream));
        else CK(cudaMemsetAsync(dp, 0, N * es, c->stream));
        for (int b = 0; b < 2; ++b)
            CK(cudaMemsetAsync(wsp<preal>(c, c->L.off_phi[b]), 0, c->L.phi_pad_elems * sizeof(preal), c->stream));
        k_phi_fill<real, TP::BX, TP::BY, TP::BZ><<<grid_for<TP>(c->P), NTP, 0, c->stream>>>(
            P, (const sreal *)scratch, wsp<preal>(c, c->L.off_phi[0]), wsp<preal>(c, c->L.off_phi[1]));
        c->launches++;
        CK(cudaGetLastError());
        c->cur = 0; c->curphi = 0;
        Fields F = fields(c, 1, 0, 0, 0);   // INIT reads no populations; writes buffer 0
        int rc = (P.grad_scheme || P.div_scheme) ? launch_main<MODE_INIT_VAR>(c, F) : launch_main<MODE_INIT>(c, F);
        if (rc) return rc;
        CK(cudaStreamSynchronize(c->stream));
        c->nsteps = 0;
        c->inited = true; c->phase = 0; c->partial = false;
        return LBM_OK;
    }

    // phase 0 of a step: K_phi (phi^{n+1} of every node, Eq.32)
    static int launch_phi(lbm_ctx *c) {
        const DevParams<real> &P = dev_params<real>(c);
        const int in = c->cur, pnew = 1 - c->curphi;
        dim3 gphi = grid_layers<TP>(c);
        if (D == 3) gphi.z = (gphi.z + PHI_NPT - 1) / PHI_NPT; else gphi.y = (gphi.y + PHI_NPT - 1) / PHI_NPT;
        if constexpr (PAIRABLE) {
            if (c->pair) {   // two x-adjacent nodes per thread (k_main_pair.cuh)
                k_phi_pair<LG, TP::BX, TP::BY, TP::BZ, PHI_NPT><<<gphi, NTP / 2, 0, c->stream>>>(
                    c->pf, (const float *)wsp<float>(c, c->L.off_g[in]), wsp<double>(c, c->L.off_phi[pnew]));
                c->launches++;
                CK(cudaGetLastError());
                return LBM_OK;
            }
        }
        k_phi<LG, real, TP::BX, TP::BY, TP::BZ, PHI_NPT><<<gphi, NTP, 0, c->stream>>>(
            P, (const sreal *)wsp<sreal>(c, c->L.off_g[in]), wsp<preal>(c, c->L.off_phi[pnew]));
        c->launches++;
        CK(cudaGetLastError());
        return LBM_OK;
    }

    // phase 1 of a step: K_main, then (flip) the buffers flip
    static int launch_collide(lbm_ctx *c, bool macro, bool flip = true) {
        const DevParams<real> &P = dev_params<real>(c);
        const int in = c->cur, out = 1 - c->cur, pnew = 1 - c->curphi, pold = c->curphi;
        Fields F = fields(c, in, out, pnew, pold);
        int rc;
        if (P.grad_scheme || P.div_scheme) {   // model variants (include/lbm.h): direct kernel; the stencil divergence reads the
            rc = LBM_OK;                       // neighbours' NEW velocity, so a velocity pass over every node comes first
            if (P.div_scheme && !P.prescribed_u) rc = launch_main<MODE_U>(c, F, pnew);
            if (!rc) rc = launch_main<MODE_STEP_VAR>(c, F, pnew);
        } else if (P.prescribed_u) rc = launch_main<MODE_STEP_PU>(c, F, pnew);   // direct kernel only
        else rc = macro ? launch_main<MODE_STEP_MACRO>(c, F, pnew) : launch_main<MODE_STEP>(c, F, pnew);
        if (rc) return rc;
        if (flip) { c->cur = out; c->curphi = pnew; c->nsteps++; }
        return LBM_OK;
    }

    // one phase on the layers [first, first + count) of the slowest axis only (lbm_step_layers, include/lbm.h)
    static int step_layers(lbm_ctx *c, int phase, int first, int count, int macro, int last) {
        if (count == 0) {   // nothing to launch: the last "part" of phase 1 still flips the buffers
            if (phase == 1 && last) { c->cur = 1 - c->cur; c->curphi = 1 - c->curphi; c->nsteps++; }
            return LBM_OK;
        }
        c->pd.s0 = c->pf.s0 = first; c->pd.s1 = c->pf.s1 = first + count;
        const int rc = phase == 0 ? launch_phi(c) : launch_collide(c, macro != 0, last != 0);
        c->pd.s0 = c->pf.s0 = 0; c->pd.s1 = c->pf.s1 = D == 3 ? c->P.nz : c->P.ny;
        return rc;
    }

    // the two phases separately, for slab contexts whose ghost layers are exchanged in between (include/lbm.h)
    static int step_phase(lbm_ctx *c, int phase, int macro) {
        return phase == 0 ? launch_phi(c) : launch_collide(c, macro != 0);
    }

    // enqueue the kernels of ONE step and flip the buffers
    static int step_once(lbm_ctx *c, bool macro, bool timed) {
        cudaEvent_t e3[3] = {nullptr, nullptr, nullptr};
        if (timed) {
            for (auto &e : e3) CK(cudaEventCreate(&e));
            CK(cudaEventRecord(e3[0], c->stream));
        }
        int rc = launch_phi(c);
        if (rc) return rc;
        if (timed) CK(cudaEventRecord(e3[1], c->stream));
        rc = launch_collide(c, macro);
        if (rc) return rc;
        if (timed) {
            CK(cudaEventRecord(e3[2], c->stream));
            for (auto e : e3) c->ev.push_back(e);
        }
        return LBM_OK;
    }

    // n steps; the last one also stores u, p, T.  On small (launch-bound) grids the plain steps are replayed from a CUDA
    // graph of two consecutive steps (the buffers alternate with period 2), captured once per context.
    static int step(lbm_ctx *c, int n) {
        if (n <= 0) return LBM_OK;
        int plain = n - 1;
        if (c->graph_ok && !c->timing && plain >= 4) {
            if (c->cur != 0) { int rc = step_once(c, false, false); if (rc) return rc; --plain; }
            if (!c->graph2) {
                const long long steps0 = c->nsteps, launches0 = c->launches;
                CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
                int rc = step_once(c, false, false);
                if (!rc) rc = step_once(c, false, false);
                cudaGraph_t g = nullptr;
                cudaError_t e = cudaStreamEndCapture(c->stream, &g);
                c->graph_launches = (int)(c->launches - launches0);
                c->nsteps = steps0; c->launches = launches0;      // nothing ran: capture only records
                if (rc) { if (g) cudaGraphDestroy(g); return rc; }
                CK(e);
                e = cudaGraphInstantiate(&c->graph2, g, 0);
                cudaGraphDestroy(g);
                CK(e);
            }
            while (plain >= 2) {
                CK(cudaGraphLaunch(c->graph2, c->stream));
                plain -= 2; c->nsteps += 2; c->launches += c->graph_launches;
            }
        }
        while (plain-- > 0) { int rc = step_once(c, false, c->timing && c->ev.size() < 3 * 4096); if (rc) return rc; }
        return step_once(c, true, c->timing && c->ev.size() < 3 * 4096);
    }

    static int read_macro(lbm_ctx *c, void *h_phi, void *h_u, void *h_p, void *h_T) {
        const size_t N = (size_t)c->L.N, es = sizeof(sreal);
        if (h_phi) {
            sreal *scratch = wsp<sreal>(c, c->L.off_scratch);
            k_phi_unpad<real, TP::BX, TP::BY, TP::BZ><<<grid_for<TP>(c->P), NTP, 0, c->stream>>>(
                dev_params<real>(c), (const preal *)wsp<preal>(c, c->L.off_phi[c->curphi]), scratch);
            c->launches++;
            CK(cudaGetLastError());
            CK(cudaMemcpyAsync(h_phi, scratch, N * es, cudaMemcpyDefault, c->stream));
        }
        if (h_u) CK(cudaMemcpyAsync(h_u, wsp<sreal>(c, c->L.off_u), 3 * N * es, cudaMemcpyDefault, c->stream));
        if (h_p) CK(cudaMemcpyAsync(h_p, wsp<sreal>(c, c->L.off_p), N * es, cudaMemcpyDefault, c->stream));
        if (h_T) CK(cudaMemcpyAsync(h_T, wsp<sreal>(c, c->L.off_T), N * es, cudaMemcpyDefault, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        return LBM_OK;
    }

    template <class L> static int read_pops_one(lbm_ctx *c, int which, int stage, const size_t (&off)[2], void *h) {
        const size_t N = (size_t)c->L.N, bytes = (size_t)L::Q * N * sizeof(sreal);
        const bool is_g = which == LBM_POPS_G;
        if (stage == LBM_STAGE_POSTCOLLISION) {
            CK(cudaMemcpyAsync(h, wsp<sreal>(c, off[c->cur]), bytes, cudaMemcpyDefault, c->stream));
            if (is_g) {   // the stored rest population carries dt/2 Pdot of its buffer (k_main.cuh): hand out g*_0 itself
                sreal *scratch = wsp<sreal>(c, c->L.off_scratch);
                k_unfold_g0<real, sreal><<<(unsigned)((N + 255) / 256), 256, 0, c->stream>>>(
                    scratch, (const sreal *)wsp<sreal>(c, off[c->cur]), (const sreal *)wsp<sreal>(c, c->L.off_pdot[c->cur]),
                    (long long)N, dev_params<real>(c).hdt);
                c->launches++;
                CK(cudaGetLastError());
                CK(cudaMemcpyAsync(h, scratch, N * sizeof(sreal), cudaMemcpyDefault, c->stream));
            }
            CK(cudaStreamSynchronize(c->stream));
            return LBM_OK;
        }
        if (c->nsteps < 1) return LBM_E_STATE;
        sreal *tmp = nullptr;
        CK(cudaMalloc(&tmp, bytes));   // debug path: own temporary, not the borrowed workspace
        k_stream_only<L, real, TP::BX, TP::BY, TP::BZ><<<grid_for<TP>(c->P), NTP, 0, c->stream>>>(
            dev_params<real>(c), (const sreal *)wsp<sreal>(c, off[1 - c->cur]), tmp, which,
            is_g ? (const sreal *)wsp<sreal>(c, c->L.off_pdot[1 - c->cur]) : (const sreal *)nullptr);
        c->launches++;
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemcpyAsync(h, tmp, bytes, cudaMemcpyDefault, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        cudaFree(tmp);
        CK(e);
        return LBM_OK;
    }

    static int read_pops(lbm_ctx *c, int which, int stage, void *h) {
        if (which == LBM_POPS_F) return read_pops_one<LF>(c, which, stage, c->L.off_f, h);
        if (which == LBM_POPS_G) return read_pops_one<LG>(c, which, stage, c->L.off_g, h);
        if (which == LBM_POPS_S) return read_pops_one<LS>(c, which, stage, c->L.off_s, h);
        return LBM_E_INVALID;
    }

    // lbm_read_pops_noalloc (noalloc.cu): the streamed populations staged in d_tmp (`cap` bytes, device memory that is not part
    // of the workspace) instead of a temporary from cudaMalloc.  Allocates nothing.
    template <class L> static int read_pops_scratch_one(lbm_ctx *c, int which, const size_t (&off)[2], void *h, void *d_tmp, size_t cap) {
        const size_t N = (size_t)c->L.N, bytes = (size_t)L::Q * N * sizeof(sreal);
        if (bytes > cap) return LBM_E_TOOLARGE;
        if (c->nsteps < 1) return LBM_E_STATE;
        sreal *tmp = static_cast<sreal *>(d_tmp);
        k_stream_only<L, real, TP::BX, TP::BY, TP::BZ><<<grid_for<TP>(c->P), NTP, 0, c->stream>>>(
            dev_params<real>(c), (const sreal *)wsp<sreal>(c, off[1 - c->cur]), tmp, which,
            which == LBM_POPS_G ? (const sreal *)wsp<sreal>(c, c->L.off_pdot[1 - c->cur]) : (const sreal *)nullptr);
        c->launches++;
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(h, tmp, bytes, cudaMemcpyDefault, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        return LBM_OK;
    }
    static int read_pops_scratch(lbm_ctx *c, int which, int stage, void *h, void *d_tmp, size_t cap) {
        if (stage == LBM_STAGE_POSTCOLLISION) return read_pops(c, which, stage, h);   // that stage never allocated
        if (which == LBM_POPS_F) return read_pops_scratch_one<LF>(c, which, c->L.off_f, h, d_tmp, cap);
        if (which == LBM_POPS_G) return read_pops_scratch_one<LG>(c, which, c->L.off_g, h, d_tmp, cap);
        if (which == LBM_POPS_S) return read_pops_scratch_one<LS>(c, which, c->L.off_s, h, d_tmp, cap);
        return LBM_E_INVALID;
    }

    static const ImplOps *ops() {
        static const ImplOps o = {&Impl::init, &Impl::step, &Impl::step_phase, &Impl::step_layers, &Impl::read_macro, &Impl::read_pops, &Impl::read_pops_scratch, T::BX, T::BY, T::BZ};
        return &o;
    }
};

}  // namespace lbm
