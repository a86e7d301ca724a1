// K_main, TMA variant: persistent CTAs (one per SM) walk over tiles of TX x TY nodes; one elected thread stages
// every input row of the NEXT tile (the pulled rows of the 33 populations, the phi^{n+1} halo rows, phi^n, Pdot) in
// shared memory with cp.async.bulk.tensor (TMA) completing on an mbarrier, while all threads compute the current
// tile from the other stage.  The pull-stream IS the TMA box coordinate: the row of direction i is fetched from
// (y - e_y, z - e_z) (wrapped by the issuing thread) starting at x0 - HALO, and read at [tx + HALO - e_x].
//   * x wrap on periodic rows: the two edge lanes fetch their wrapped value with one global load per direction;
//   * tiles that touch a non-periodic face (walls, heated plate, open face) take the direct gather path
//     (SrcGlobal<BC = true>) inside the same kernel -- the choice is tile-uniform, so no warp diverges.
// Arithmetic is node_update() of k_main.cuh, shared with the direct variant.
#pragma once

#include <cuda.h>

#include <cstdint>

#include "k_main.cuh"

namespace lbm {

// ---- PTX wrappers -----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}

// ---- tile configuration -----------------------------------------------------------------------------------------
template <class LF, class LG, class LS, class real> struct TmaCfg {
    static constexpr int D = LF::D;
    static constexpr int TX = 128, TY = 2, NS = 2;
    static constexpr int NT = TX * TY;
    static constexpr int EPB = 16 / (int)sizeof(real);                       // elements per 16 bytes
    static constexpr int HALO = EPB;                                         // TMA box starts must be 16-byte aligned (measured:
                                                                             // an odd fp64 start coordinate traps), so the halo is 16 bytes
    static constexpr int BOXX = TX + 2 * HALO;
    static constexpr int RS = (BOXX * (int)sizeof(real) + 127) / 128 * 128 / (int)sizeof(real);   // row stride (elements), 128-byte rows
    static constexpr int NPOP = LF::Q + LG::Q + LS::Q;
    static constexpr int NZ3 = D == 3 ? 3 : 1;
    static constexpr int ROW_F = 0, ROW_G = LF::Q * TY, ROW_S = (LF::Q + LG::Q) * TY;
    static constexpr int ROW_PHI = NPOP * TY;                                // NZ3 * (TY + 2) rows
    static constexpr int ROW_PHIOLD = ROW_PHI + NZ3 * (TY + 2);
    static constexpr int ROW_PDOT = ROW_PHIOLD + TY;
    static constexpr int NROWS = ROW_PDOT + TY;
    static constexpr uint32_t TX_BYTES = (uint32_t)NROWS * BOXX * sizeof(real);
    static constexpr size_t STAGE_BYTES = (size_t)NROWS * RS * sizeof(real);
    static constexpr size_t SMEM_BYTES = NS * STAGE_BYTES + 128;             // + mbarriers
};

struct TmaMaps {
    CUtensorMap f, g, s;        // [x][y][z][q] of the input (post-collision, previous level) populations
    CUtensorMap phi_new, phi_old;   // padded phi buffers
    CUtensorMap pdot;
};

// Source of one node's inputs from the shared-memory stage.
template <class LF, class LG, class LS, class real> struct SrcTma {
    using C = TmaCfg<LF, LG, LS, real>;
    const DevParams<real> &P;
    const DevFields<real> &Fd;
    const NodeGeom &g;
    const real *st;    // stage base
    int tx, ry;
    __device__ __forceinline__ SrcTma(const DevParams<real> &P_, const DevFields<real> &Fd_, const NodeGeom &g_,
                                      const real *st_, int tx_, int ry_)
        : P(P_), Fd(Fd_), g(g_), st(st_), tx(tx_), ry(ry_) {}
    __device__ __forceinline__ void pops_ready() const {}
    __device__ __forceinline__ void f_ready() const {}
    __device__ __forceinline__ void phi_ready() const {}
    __device__ __forceinline__ real phi(int dx, int dy, int dz) const {
        const int row = C::ROW_PHI + (C::D == 3 ? (dz + 1) : 0) * (C::TY + 2) + ry + 1 + dy;
        return st[row * C::RS + tx + C::HALO + dx];
    }
    __device__ __forceinline__ real phi_old() const { return st[(C::ROW_PHIOLD + ry) * C::RS + tx + C::HALO]; }
    __device__ __forceinline__ real pdot_old() const { return st[(C::ROW_PDOT + ry) * C::RS + tx + C::HALO]; }
    template <class L, int ROW0, int I, bool AGAIN>
    __device__ __forceinline__ real get(const real *__restrict__ gsrc) const {
        constexpr int ex = L::ex(I);
        const real *q = st + ((ROW0 + I * C::TY + ry) * C::RS + tx + C::HALO - ex);
        real v = AGAIN ? *reinterpret_cast<const volatile real *>(q) : *q;   // volatile: a real second read, not a held register
        if constexpr (ex != 0) {
            // periodic x wrap: the halo element of an edge tile is outside the array (TMA fills zeros)
            if (ex > 0 ? g.lo[0] : g.hi[0])
                v = __ldg(gsrc + (unsigned)I * (unsigned)P.N + g.sz[L::ez(I) + 1] + g.sy[L::ey(I) + 1] + g.sx[ex + 1]);
        }
        return v;
    }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real f() const { return get<LF, C::ROW_F, I, AGAIN>(Fd.f_in); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real gg() const { return get<LG, C::ROW_G, I, AGAIN>(Fd.g_in); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real s() const { return get<LS, C::ROW_S, I, AGAIN>(Fd.s_in); }
};

// tile index -> origin; tiles are enumerated x-fastest, then y, then z
template <class C, class real>
__device__ __forceinline__ void tile_origin(const DevParams<real> &P, long long tile, int nxt, int nyt, int &x0, int &y0, int &z0) {
    const int xt = (int)(tile % nxt);
    const long long r = tile / nxt;
    x0 = xt * C::TX;
    y0 = (int)(r % nyt) * C::TY;
    z0 = (int)(r / nyt);
}

// one thread: issue every row of tile (x0, y0, z0) into stage `dst`, completing on `bar`
template <class LF, class LG, class LS, class real>
__device__ __forceinline__ void issue_tile(const DevParams<real> &P, const TmaMaps &M, uint32_t dst, uint32_t bar,
                                           int x0, int y0, int z0) {
    using C = TmaCfg<LF, LG, LS, real>;
    constexpr uint32_t RSB = C::RS * sizeof(real);
    mbar_expect_tx(bar, C::TX_BYTES);
    auto wrap = [](int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); };
#pragma unroll
    for (int ry = 0; ry < C::TY; ++ry) {
        const int y = y0 + ry;
        const bool row_ok = y < P.ny;
        auto pops = [&](auto lat, const CUtensorMap *map, int row0) {
            using L = decltype(lat);
            static_for<L::Q>([&](auto ic) {
                constexpr int I = decltype(ic)::value;
                const int ys = row_ok ? wrap(y - L::ey(I), P.ny) : y;       // rows past the end: out of bounds -> zeros
                const int zs = wrap(z0 - L::ez(I), P.nz);
                tma_load_4d(dst + (uint32_t)(row0 + I * C::TY + ry) * RSB, map, bar, x0 - C::HALO, ys, zs, I);
            });
        };
        pops(LF{}, &M.f, C::ROW_F);
        pops(LG{}, &M.g, C::ROW_G);
        pops(LS{}, &M.s, C::ROW_S);
        tma_load_3d(dst + (uint32_t)(C::ROW_PHIOLD + ry) * RSB, &M.phi_old, bar, x0, y + 1, z0 + P.pz);
        tma_load_3d(dst + (uint32_t)(C::ROW_PDOT + ry) * RSB, &M.pdot, bar, x0 - C::HALO, y, z0);
    }
#pragma unroll
    for (int dz = 0; dz < C::NZ3; ++dz)
#pragma unroll
        for (int r = 0; r < C::TY + 2; ++r)      // padded rows y0-1 .. y0+TY  ->  padded index y0 .. y0+TY+1
            tma_load_3d(dst + (uint32_t)(C::ROW_PHI + dz * (C::TY + 2) + r) * RSB, &M.phi_new, bar, x0, y0 + r,
                        z0 + P.pz + (C::D == 3 ? dz - 1 : 0));
}

template <class LF, class LG, class LS, class real, int MODE>
__global__ void __launch_bounds__(TmaCfg<LF, LG, LS, real>::NT, 1)
k_main_tma(const DevParams<real> P, const DevFields<real> Fd, const __grid_constant__ TmaMaps M, long long ntiles,
           int nxt, int nyt) {
    using C = TmaCfg<LF, LG, LS, real>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    real *stage0 = reinterpret_cast<real *>(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem_raw + C::NS * C::STAGE_BYTES);
    const int t = threadIdx.x;
    const int tx = t % C::TX, ry = t / C::TX;

    if (t == 0) {
#pragma unroll
        for (int s = 0; s < C::NS; ++s) mbar_init(smem_u32(&bars[s]), 1);
        fence_mbar_init();
        fence_proxy_async();
    }
    __syncthreads();

    auto is_direct = [&](long long tile) {
        int x0, y0, z0;
        tile_origin<C>(P, tile, nxt, nyt, x0, y0, z0);
        return tile_touches_bc(P, x0, y0, z0, C::TX, C::TY, 1);
    };

    // issue cursor (thread 0 only): next tile of this CTA that goes through TMA
    long long issue_tile_id = blockIdx.x;
    int issued = 0;
    auto issue_next = [&]() {
        while (issue_tile_id < ntiles && is_direct(issue_tile_id)) issue_tile_id += gridDim.x;
        if (issue_tile_id < ntiles) {
            int x0, y0, z0;
            tile_origin<C>(P, issue_tile_id, nxt, nyt, x0, y0, z0);
            const int s = issued % C::NS;
            issue_tile<LF, LG, LS, real>(P, M, smem_u32(smem_raw + (size_t)s * C::STAGE_BYTES), smem_u32(&bars[s]), x0, y0, z0);
            ++issued;
            issue_tile_id += gridDim.x;
        }
    };
    if (t == 0) {
#pragma unroll
        for (int s = 0; s < C::NS; ++s) issue_next();
    }

    int consumed = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        int x0, y0, z0;
        tile_origin<C>(P, tile, nxt, nyt, x0, y0, z0);
        const int x = x0 + tx, y = y0 + ry, z = z0;
        const bool active = x < P.nx && y < P.ny;
        if (tile_touches_bc(P, x0, y0, z0, C::TX, C::TY, 1)) {
            if (active) {
                const NodeGeom g = make_geom(P, x, y, z);
                const SrcGlobal<LF, LG, LS, real, true> src(P, Fd, g);
                node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
            }
            continue;
        }
        const int s = consumed % C::NS;
        mbar_wait(smem_u32(&bars[s]), (uint32_t)((consumed / C::NS) & 1));
        if (active) {
            const NodeGeom g = make_geom(P, x, y, z);
            const SrcTma<LF, LG, LS, real> src(P, Fd, g, stage0 + (size_t)s * (C::STAGE_BYTES / sizeof(real)), tx, ry);
            node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
        }
        ++consumed;
        __syncthreads();                 // every thread is done reading stage s
        if (t == 0) {
            fence_proxy_async();         // order those generic-proxy reads before the async-proxy refill
            issue_next();
        }
    }
}

}  // namespace lbm
