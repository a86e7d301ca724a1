// K_main, gather variant with EVERY input of the node staged in shared memory: the phi^{n+1} halo tile by one TMA box per CTA
// (as k_main_phitma.cuh) and the pulled f and s populations (26 in 3D), phi^n and Pdot by per-thread asynchronous copies
// (cp.async -> LDGSTS) into the thread's own column of a [value][thread] array.  All of a thread's loads are in flight at once
// without occupying registers (Little's law: 16 warps x 32 lanes x 28 x 8 B = 115 KB in flight per SM), and the second read of every
// population at collision time is a shared-memory load instead of an L2 round trip (the 200 KB L1 does not hold the
// 16 x 18 KB working set of the gather kernel: its measured L1 hit rate is 5%).  Tiles that touch a non-periodic face take
// the gather path of k_main_phitma.cuh (boundary rules select other addresses); the choice is tile-uniform.
#pragma once

#include "k_main_phitma.cuh"

namespace lbm {

// shared-memory carve-up of one CTA of NT threads
// STAGE_G: g is read once (at its collision), so staging it only buys the early issue (measured: no gain; off).
template <class LF, class LG, class LS, class sreal, class preal, int BX, int BY, int BZ, bool STAGE_G_ = false> struct SmemCfg {
    using TC = PhiTileCfg<preal, LF::D, BX, BY, BZ>;
    static constexpr int NT = BX * BY * BZ;
    static constexpr bool STAGE_G = STAGE_G_;
    static constexpr int QT = LF::Q + LS::Q + (STAGE_G ? LG::Q : 0);
    static constexpr int OFF_F = 0, OFF_S = LF::Q, OFF_G = LF::Q + LS::Q, OFF_PDOT = QT;   // sreal slots
    static constexpr size_t TILE_BYTES = ((size_t)TC::BYTES + 127) / 128 * 128;
    static constexpr size_t PHIOLD_BYTES = (size_t)NT * sizeof(preal);
    static constexpr size_t POPS_BYTES = (size_t)(QT + 1) * NT * sizeof(sreal);
    static constexpr size_t BYTES = TILE_BYTES + PHIOLD_BYTES + POPS_BYTES + 16;   // + the mbarrier
};

template <class LF, class LG, class LS, class real, class C, class Fields> struct SrcSmem {
    using sreal = typename Fields::sreal;
    using preal = typename Fields::preal;
    using TC = typename C::TC;
    const DevParams<real> &P;
    const Fields &Fd;
    const NodeGeom &g;
    const preal *tile;      // the node's own element in the phi tile
    const preal *phiold;    // this thread's slot
    const sreal *col;       // this thread's column: value k at col[k * NT]
    uint32_t bar;
    __device__ __forceinline__ SrcSmem(const DevParams<real> &P_, const Fields &Fd_, const NodeGeom &g_, const preal *tile_base,
                                       const preal *phiold_base, const sreal *pops_base, uint32_t bar_, int t, int tx, int ty, int tz)
        : P(P_), Fd(Fd_), g(g_), bar(bar_) {
        tile = tile_base + ((LF::D == 3 ? tz + 1 : 0) * TC::BOXY + ty + 1) * TC::BOXX + tx + TC::EPB;
        phiold = phiold_base + t;
        col = pops_base + t;
    }
    // issue every copy of this node; nothing is waited for here
    __device__ __forceinline__ void prefetch() const {
        const unsigned N = (unsigned)P.N;
        const uint32_t c0 = smem_u32(col);
        constexpr uint32_t STEP = (uint32_t)(C::NT * sizeof(sreal));
        static_for<LS::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            cp_async_val(c0 + (uint32_t)(C::OFF_S + I) * STEP, Fd.s_in + pull_offset<LS, I>(N, g));
        });
        cp_async_val(c0 + (uint32_t)C::OFF_PDOT * STEP, Fd.pdot_in + g.n);
        const unsigned pcoff = ((unsigned)(g.z + P.pz) * (unsigned)P.ppy + (unsigned)(g.y + 1)) * (unsigned)P.ppx + (unsigned)(g.x + P.xpad);
        cp_async_val(smem_u32(phiold), Fd.phi_old + pcoff);
        cp_async_commit();   // group 1: what the stencil and closure phase needs (s, Pdot, phi^n)
        static_for<LF::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            cp_async_val(c0 + (uint32_t)(C::OFF_F + I) * STEP, Fd.f_in + pull_offset<LF, I>(N, g));
        });
        if constexpr (C::STAGE_G) {
            static_for<LG::Q>([&](auto ic) {
                constexpr int I = decltype(ic)::value;
                cp_async_val(c0 + (uint32_t)(C::OFF_G + I) * STEP, Fd.g_in + pull_offset<LG, I>(N, g));
            });
        }
        cp_async_commit();   // group 2: f (and g), first needed by the moments
    }
    // own copies only: no CTA barrier needed, nobody else reads the column
    __device__ __forceinline__ void pops_ready() const { cp_async_wait_1(); }
    __device__ __forceinline__ void f_ready() const { cp_async_wait_all(); }
    __device__ __forceinline__ void phi_ready() const { mbar_wait(bar, 0); }
    __device__ __forceinline__ preal phi(int dx, int dy, int dz) const { return tile[dx + dy * TC::BOXX + dz * (TC::BOXX * TC::BOXY)]; }
    __device__ __forceinline__ preal phi_old() const { return *phiold; }
    __device__ __forceinline__ real pdot_old() const { return real(col[C::OFF_PDOT * C::NT]); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real f() const { return real(col[(C::OFF_F + I) * C::NT]); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real s() const { return real(col[(C::OFF_S + I) * C::NT]); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real gg() const {
        if constexpr (C::STAGE_G) return real(col[(C::OFF_G + I) * C::NT]);
        else return real(__ldg(Fd.g_in + pull_offset<LG, I>((unsigned)P.N, g)));
    }
};

// one tile of BX x BY x BZ nodes with origin (x0, y0, z0); smem_raw: SmemCfg::BYTES bytes of dynamic shared memory
template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int BZ, bool STAGE_G = false, class Fields>
__device__ __forceinline__ void main_tile_smem(const DevParams<real> &P, const Fields &Fd, const CUtensorMap *phi_map,
                                               unsigned char *smem_raw, int x0, int y0, int z0) {
    using sreal = typename Fields::sreal;
    using preal = typename Fields::preal;
    using C = SmemCfg<LF, LG, LS, sreal, preal, BX, BY, BZ, STAGE_G>;
    using TC = typename C::TC;
    preal *tile = reinterpret_cast<preal *>(smem_raw);
    preal *phiold = reinterpret_cast<preal *>(smem_raw + C::TILE_BYTES);
    sreal *pops = reinterpret_cast<sreal *>(smem_raw + C::TILE_BYTES + C::PHIOLD_BYTES);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + C::TILE_BYTES + C::PHIOLD_BYTES + C::POPS_BYTES);
    const int t = threadIdx.x;
    const int tx = t % BX, ty = (t / BX) % BY, tz = t / (BX * BY);
    const uint32_t bar_a = smem_u32(bar);
    if (t == 0) {
        mbar_init(bar_a, 1);
        fence_mbar_init();
        fence_proxy_async();
    }
    const int x = x0 + tx, y = y0 + ty, z = z0 + tz;
    const bool active = node_active<LF::D>(P, x, y, z);
    const bool bc = tile_touches_bc(P, x0, y0, z0, BX, BY, BZ);
    NodeGeom g;
    if (active) {
        g = make_geom(P, x, y, z);
        if (!bc) {
            const SrcSmem<LF, LG, LS, real, C, Fields> src(P, Fd, g, tile, phiold, pops, bar_a, t, tx, ty, tz);
            src.prefetch();   // before the barrier below: the copies fly while the CTA assembles
        }
    }
    if (t == 0) {
        // phi^{n+1} is K_phi's output, the only input the preceding launch writes: with programmatic dependent launch this CTA
        // may be running before K_phi has finished, its population copies (above) already in flight
        pdl_wait();
        mbar_expect_tx(bar_a, TC::BYTES);
        tma_load_3d(smem_u32(tile), phi_map, bar_a, x0, y0, LF::D == 3 ? z0 : 0);
    }
    __syncthreads();   // the mbarrier is initialised before anybody waits on it
    if (!active) return;
    if (bc) {
        const SrcGlobalPhiSmem<LF, LG, LS, real, true, TC, Fields> src(P, Fd, g, tile, bar_a, tx, ty, tz);
        node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
    } else {
        const SrcSmem<LF, LG, LS, real, C, Fields> src(P, Fd, g, tile, phiold, pops, bar_a, t, tx, ty, tz);
        node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
    }
}

template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int BZ, int MINB, class Fields>
__global__ void __launch_bounds__(BX *BY *BZ, MINB)
k_main_smem(const DevParams<real> P, const Fields Fd, const __grid_constant__ CUtensorMap phi_map) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    int y0, z0;
    tile_origin<LF::D>(P, BY, BZ, y0, z0);
    main_tile_smem<LF, LG, LS, real, MODE, BX, BY, BZ>(P, Fd, &phi_map, smem_raw, blockIdx.x * BX, y0, z0);
}

}  // namespace lbm
