// K_main, gather variant with the phi^{n+1} halo tile staged in shared memory by ONE TMA box per CTA
// (cp.async.bulk.tensor.3d -> UTMALDG, completing on an mbarrier).  The 19 (3D) / 9 (2D) stencil reads of every
// node become shared-memory loads; the populations are gathered from global memory as in k_main_direct.
// The padded phi array has materialised ghost layers and a 16-byte x offset (xpad), so the box
// [x0 - EPB, x0 + BX + EPB) x [y0 - 1, y0 + BY] x [z0 - 1, z0 + BZ] always starts 16-byte aligned and never needs wrap logic.
//
// The tile bodies are device functions taking the tile origin, so that other kernels can run a tile at a place of their own.
#pragma once

#include "k_main.cuh"
#include "ptx.cuh"

namespace lbm {

template <class real, int D, int BX, int BY, int BZ> struct PhiTileCfg {
    static constexpr int EPB = 16 / (int)sizeof(real);
    static constexpr int BOXX = BX + 2 * EPB;
    static constexpr int BOXY = BY + 2;
    static constexpr int BOXZ = D == 3 ? BZ + 2 : 1;
    static constexpr int ELEMS = BOXX * BOXY * BOXZ;
    static constexpr uint32_t BYTES = (uint32_t)ELEMS * sizeof(real);
};

template <class LF, class LG, class LS, class real, bool BC, class TC, class Fields> struct SrcGlobalPhiSmem {
    using preal = typename Fields::preal;
    const DevParams<real> &P;
    const Fields &Fd;
    const NodeGeom &g;
    const preal *tile;    // the node's own element in the shared-memory tile
    uint32_t bar;
    unsigned pcoff;
    __device__ __forceinline__ SrcGlobalPhiSmem(const DevParams<real> &P_, const Fields &Fd_, const NodeGeom &g_,
                                                const preal *tile_base, uint32_t bar_, int tx, int ty, int tz)
        : P(P_), Fd(Fd_), g(g_), bar(bar_) {
        tile = tile_base + ((LF::D == 3 ? tz + 1 : 0) * TC::BOXY + ty + 1) * TC::BOXX + tx + TC::EPB;
        pcoff = ((unsigned)(g.z + P.pz) * (unsigned)P.ppy + (unsigned)(g.y + 1)) * (unsigned)P.ppx + (unsigned)(g.x + P.xpad);
    }
    __device__ __forceinline__ void pops_ready() const {}
    __device__ __forceinline__ void f_ready() const {}
    __device__ __forceinline__ void phi_ready() const { mbar_wait(bar, 0); }
    __device__ __forceinline__ preal phi(int dx, int dy, int dz) const { return tile[dx + dy * TC::BOXX + dz * (TC::BOXX * TC::BOXY)]; }
    __device__ __forceinline__ preal phi_old() const { return __ldg(Fd.phi_old + pcoff); }
    __device__ __forceinline__ real pdot_old() const { return real(Fd.pdot_in[g.n]); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real f() const { return pull_one<LF, I, real, BC, AGAIN>(Fd.f_in, (unsigned)P.N, g, P.bc_f, P.bc_p); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real s() const { return pull_one<LS, I, real, BC, AGAIN>(Fd.s_in, (unsigned)P.N, g, P.bc_s, P.bc_T); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real gg() const { return pull_one<LG, I, real, BC, AGAIN>(Fd.g_in, (unsigned)P.N, g, P.bc_g, P.bc_phi); }
};

// shared memory of one CTA: the phi tile and its mbarrier
template <class preal, class TC> struct PhiTileSmem {
    static constexpr size_t TILE_BYTES = ((size_t)TC::BYTES + 127) / 128 * 128;
    static constexpr size_t BYTES = TILE_BYTES + 16;
};

// one tile of BX x BY x BZ nodes with origin (x0, y0, z0); smem_raw: PhiTileSmem::BYTES bytes, 128-byte aligned
template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int BZ, class Fields>
__device__ __forceinline__ void main_tile_phitma(const DevParams<real> &P, const Fields &Fd, const CUtensorMap *phi_map,
                                                 unsigned char *smem_raw, int x0, int y0, int z0) {
    using preal = typename Fields::preal;
    using TC = PhiTileCfg<preal, LF::D, BX, BY, BZ>;
    using SM = PhiTileSmem<preal, TC>;
    preal *tile = reinterpret_cast<preal *>(smem_raw);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + SM::TILE_BYTES);
    const int t = threadIdx.x;
    const int tx = t % BX, ty = (t / BX) % BY, tz = t / (BX * BY);
    const uint32_t bar_a = smem_u32(bar);
    if (t == 0) {
        mbar_init(bar_a, 1);
        fence_mbar_init();
        fence_proxy_async();
        pdl_wait();   // phi^{n+1} is K_phi's output: the only input of this kernel that the preceding launch writes
        mbar_expect_tx(bar_a, TC::BYTES);
        // padded coordinates of node (x0 - EPB, y0 - 1, z0 - 1): (x0, y0, z0 + pz - 1)
        tma_load_3d(smem_u32(tile), phi_map, bar_a, x0, y0, LF::D == 3 ? z0 : 0);
    }
    __syncthreads();   // the barrier is initialised before anybody waits on it
    const int x = x0 + tx, y = y0 + ty, z = z0 + tz;
    if (!node_active<LF::D>(P, x, y, z)) return;
    const NodeGeom g = make_geom(P, x, y, z);
    if (tile_touches_bc(P, x0, y0, z0, BX, BY, BZ)) {
        const SrcGlobalPhiSmem<LF, LG, LS, real, true, TC, Fields> src(P, Fd, g, tile, bar_a, tx, ty, tz);
        node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
    } else {
        const SrcGlobalPhiSmem<LF, LG, LS, real, false, TC, Fields> src(P, Fd, g, tile, bar_a, tx, ty, tz);
        node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
    }
}

template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int BZ, int MINB, class Fields>
__global__ void __launch_bounds__(BX *BY *BZ, MINB)
k_main_phitma(const DevParams<real> P, const Fields Fd, const __grid_constant__ CUtensorMap phi_map) {
    using preal = typename Fields::preal;
    using SM = PhiTileSmem<preal, PhiTileCfg<preal, LF::D, BX, BY, BZ>>;
    __shared__ __align__(128) unsigned char smem_raw[SM::BYTES];
    int y0, z0;
    tile_origin<LF::D>(P, BY, BZ, y0, z0);
    main_tile_phitma<LF, LG, LS, real, MODE, BX, BY, BZ>(P, Fd, &phi_map, smem_raw, blockIdx.x * BX, y0, z0);
}

}  // namespace lbm
