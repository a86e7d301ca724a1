// K_main in single precision with TWO x-adjacent nodes per thread (3D, float populations, double phi).  The float kernels with one
// node per thread are instruction-bound, not HBM-bound (issue slots 54% busy at 71% of the DRAM peak, profiles/r1_kernels_full.md):
// as many warp instructions per node as in double for half the bytes.  A thread that carries the pair (x, x + 1), x even, is the
// double-precision thread again: every value it holds is 8 bytes (an f2, pairs.cuh), populations whose link has e_x = 0 arrive
// and leave as ONE 8-byte access, and the arithmetic is the packed f32x2 instructions of sm_100 (FFMA2 / FADD2 / FMUL2) -- node_update
// (k_main.cuh) is instantiated with real = f2, nothing of the method is restated here.  The phi halo tile is the TMA box of
// k_main_phitma.cuh.  Tiles that touch a non-periodic face run the one-node code twice per thread (tile-uniform choice).
#pragma once

#include "k_main_smem.cuh"
#include "k_phi.cuh"
#include "pairs.cuh"

namespace lbm {

// geometry of the pair (x, x + 1): rows and planes are shared, the x sources of the two nodes differ
struct NodeGeom2 {
    unsigned n;        // linear index of the first node (even)
    unsigned x;
    unsigned sxm;      // source of the FIRST node for e_x = +1: x - 1, wrapped   (the second node's is x)
    unsigned sxp;      // source of the SECOND node for e_x = -1: x + 2, wrapped  (the first node's is x + 1)
    unsigned sy[3];    // (y - e_y wrapped) * nx
    unsigned sz[3];    // (z - e_z wrapped) * nx * ny
};

__device__ __forceinline__ NodeGeom2 make_geom2(const DevParams<float> &P, int x, int y, int z) {
    NodeGeom2 g;
    const unsigned row = (unsigned)P.nx, plane = (unsigned)P.nx * (unsigned)P.ny;
    g.x = (unsigned)x;
    g.n = (unsigned)z * plane + (unsigned)y * row + (unsigned)x;
    g.sxm = x == 0 ? (unsigned)(P.nx - 1) : (unsigned)(x - 1);
    g.sxp = x + 2 >= P.nx ? 0u : (unsigned)(x + 2);
    g.sy[0] = (unsigned)(y == P.ny - 1 ? 0 : y + 1) * row;  g.sy[1] = (unsigned)y * row;
    g.sy[2] = (unsigned)(y == 0 ? P.ny - 1 : y - 1) * row;
    g.sz[0] = (unsigned)(z == P.nz - 1 ? 0 : z + 1) * plane;  g.sz[1] = (unsigned)z * plane;
    g.sz[2] = (unsigned)(z == 0 ? P.nz - 1 : z - 1) * plane;
    return g;
}

__device__ __forceinline__ float2 ld_again2(const float *p) {   // see ld_again (kernels.cuh)
    float2 v;
    asm volatile("ld.global.nc.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// pull-stream direction I for the pair (periodic wrap only): one 8-byte load when the link does not move in x
template <class L, int I, bool AGAIN> __device__ __forceinline__ f2 pull_pair(const float *__restrict__ src, unsigned N, const NodeGeom2 &g) {
    const unsigned base = (unsigned)I * N + g.sz[L::ez(I) + 1] + g.sy[L::ey(I) + 1];
    if constexpr (L::ex(I) == 0) {
        const float *p = src + (base + g.x);
        const float2 v = AGAIN ? ld_again2(p) : __ldg(reinterpret_cast<const float2 *>(p));
        return f2(v.x, v.y);
    } else if constexpr (L::ex(I) > 0) {
        return f2(ld_pop<AGAIN, float>(src + (base + g.sxm)), ld_pop<AGAIN, float>(src + (base + g.x)));
    } else {
        return f2(ld_pop<AGAIN, float>(src + (base + g.x + 1u)), ld_pop<AGAIN, float>(src + (base + g.sxp)));
    }
}

template <class LF, class LG, class LS, class TC, class Fields> struct SrcPair {
    const DevParams<float> &P;
    const Fields &Fd;
    const NodeGeom2 &g;
    const double *tile;   // the first node's own element in the shared-memory phi tile
    uint32_t bar;
    unsigned pcoff;
    __device__ __forceinline__ SrcPair(const DevParams<float> &P_, const Fields &Fd_, const NodeGeom2 &g_, const double *tile_base,
                                       uint32_t bar_, int x, int y, int z, int tx, int ty, int tz)
        : P(P_), Fd(Fd_), g(g_), bar(bar_) {
        tile = tile_base + ((tz + 1) * TC::BOXY + ty + 1) * TC::BOXX + tx + TC::EPB;
        pcoff = ((unsigned)(z + P.pz) * (unsigned)P.ppy + (unsigned)(y + 1)) * (unsigned)P.ppx + (unsigned)(x + P.xpad);
    }
    __device__ __forceinline__ void pops_ready() const {}
    __device__ __forceinline__ void f_ready() const {}
    __device__ __forceinline__ void phi_ready() const { mbar_wait(bar, 0); }
    __device__ __forceinline__ d2 phi(int dx, int dy, int dz) const {
        const double *p = tile + (dx + dy * TC::BOXX + dz * (TC::BOXX * TC::BOXY));
        if ((dx & 1) == 0) {   // the first node sits on an even element of the tile (EPB = 2, x even): 16-byte aligned
            const double2 v = *reinterpret_cast<const double2 *>(p);
            return d2(v.x, v.y);
        }
        return d2(p[0], p[1]);
    }
    __device__ __forceinline__ d2 phi_old() const {
        const double2 v = __ldg(reinterpret_cast<const double2 *>(Fd.phi_old + pcoff));
        return d2(v.x, v.y);
    }
    __device__ __forceinline__ f2 pdot_old() const {
        const float2 v = __ldg(reinterpret_cast<const float2 *>(Fd.pdot_in + g.n));
        return f2(v.x, v.y);
    }
    template <int I, bool AGAIN = false> __device__ __forceinline__ f2 f() const { return pull_pair<LF, I, AGAIN>(Fd.f_in, (unsigned)P.N, g); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ f2 s() const { return pull_pair<LS, I, AGAIN>(Fd.s_in, (unsigned)P.N, g); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ f2 gg() const { return pull_pair<LG, I, AGAIN>(Fd.g_in, (unsigned)P.N, g); }
};

// ---- the same with the pair's f, s and g values and Pdot staged in shared memory by per-thread cp.async (as k_main_smem.cuh):
// 16 warps per SM holding their loads in registers leave the memory system idle (measured: 63% of the DRAM peak, issue slots 30%
// busy, 8 long-scoreboard stalls per issue); staged, all 48 copies of a pair are in flight at once.  Unlike in double precision,
// staging g pays here (K_main 1.549 -> 1.522 ms on config 4): read as plain loads at their collision, the last thing a thread
// does, their latency is exposed with nothing left to overlap it.
template <class LF, class LG, class LS, int BX, int BY, int BZ> struct PairSmemCfg {
    using TC = PhiTileCfg<double, 3, BX, BY, BZ>;
    static constexpr int NT = BX / 2 * BY * BZ;
    static constexpr int QT = LF::Q + LS::Q + LG::Q;
    static constexpr int OFF_F = 0, OFF_S = LF::Q, OFF_G = LF::Q + LS::Q, OFF_PDOT = QT;   // float2 slots
    static constexpr size_t TILE_BYTES = ((size_t)TC::BYTES + 127) / 128 * 128;
    // phi^n is NOT staged (it rides in registers from before the CTA barrier): four CTAs fit the 196 KB shared-memory configuration
    // without it, not with it
    static constexpr size_t POPS_BYTES = (size_t)(QT + 1) * NT * sizeof(float2);
    static constexpr size_t BYTES = TILE_BYTES + POPS_BYTES + 16;   // + the mbarrier
};

__device__ __forceinline__ void cp_async_8(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}

template <class LF, class LG, class LS, class C, class Fields> struct SrcPairSmem {
    using TC = typename C::TC;
    const DevParams<float> &P;
    const Fields &Fd;
    const NodeGeom2 &g;
    const double *tile;      // the first node's own element in the phi tile
    const float2 *col;       // this thread's column: value k at col[k * NT]
    uint32_t bar;
    double2 po;              // phi^n of the pair
    __device__ __forceinline__ SrcPairSmem(const DevParams<float> &P_, const Fields &Fd_, const NodeGeom2 &g_, const double *tile_base,
                                           const float2 *pops_base, uint32_t bar_, int t, int tx, int ty, int tz, double2 po_)
        : P(P_), Fd(Fd_), g(g_), bar(bar_), po(po_) {
        tile = tile_base + ((tz + 1) * TC::BOXY + ty + 1) * TC::BOXX + tx + TC::EPB;
        col = pops_base + t;
    }
    // the two values of direction I into one float2 slot: one 8-byte copy, or two 4-byte copies when the link moves in x
    template <class L, int I> __device__ __forceinline__ void copy_pair(uint32_t dst, const float *__restrict__ src, unsigned N) const {
        const unsigned base = (unsigned)I * N + g.sz[L::ez(I) + 1] + g.sy[L::ey(I) + 1];
        if constexpr (L::ex(I) == 0) cp_async_8(dst, src + (base + g.x));
        else if constexpr (L::ex(I) > 0) { cp_async_val(dst, src + (base + g.sxm)); cp_async_val(dst + 4, src + (base + g.x)); }
        else { cp_async_val(dst, src + (base + g.x + 1u)); cp_async_val(dst + 4, src + (base + g.sxp)); }
    }
    __device__ __forceinline__ void prefetch() const {
        const unsigned N = (unsigned)P.N;
        const uint32_t c0 = smem_u32(col);
        constexpr uint32_t STEP = (uint32_t)(C::NT * sizeof(float2));
        static_for<LS::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            copy_pair<LS, I>(c0 + (uint32_t)(C::OFF_S + I) * STEP, Fd.s_in, N);
        });
        cp_async_8(c0 + (uint32_t)C::OFF_PDOT * STEP, Fd.pdot_in + g.n);
        cp_async_commit();   // group 1: what the stencil and closure phase needs (s, Pdot)
        static_for<LF::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            copy_pair<LF, I>(c0 + (uint32_t)(C::OFF_F + I) * STEP, Fd.f_in, N);
        });
        static_for<LG::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            copy_pair<LG, I>(c0 + (uint32_t)(C::OFF_G + I) * STEP, Fd.g_in, N);
        });
        cp_async_commit();   // group 2: f and g, first needed by the moments
    }
    __device__ __forceinline__ void pops_ready() const { cp_async_wait_1(); }
    __device__ __forceinline__ void f_ready() const { cp_async_wait_all(); }
    __device__ __forceinline__ void phi_ready() const { mbar_wait(bar, 0); }
    __device__ __forceinline__ d2 phi(int dx, int dy, int dz) const {
        const double *p = tile + (dx + dy * TC::BOXX + dz * (TC::BOXX * TC::BOXY));
        if ((dx & 1) == 0) {
            const double2 v = *reinterpret_cast<const double2 *>(p);
            return d2(v.x, v.y);
        }
        return d2(p[0], p[1]);
    }
    __device__ __forceinline__ d2 phi_old() const { return d2(po.x, po.y); }
    __device__ __forceinline__ f2 pdot_old() const { const float2 v = col[C::OFF_PDOT * C::NT]; return f2(v.x, v.y); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ f2 f() const { const float2 v = col[(C::OFF_F + I) * C::NT]; return f2(v.x, v.y); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ f2 s() const { const float2 v = col[(C::OFF_S + I) * C::NT]; return f2(v.x, v.y); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ f2 gg() const { const float2 v = col[(C::OFF_G + I) * C::NT]; return f2(v.x, v.y); }
};

template <class LF, class LG, class LS, int MODE, int BX, int BY, int BZ, int MINB, class Fields>
__global__ void __launch_bounds__(BX / 2 * BY * BZ, MINB)
k_main_pair_smem(const DevParams<float> P, const DevParams<f2> P2, const Fields Fd, const __grid_constant__ CUtensorMap phi_map) {
    using C = PairSmemCfg<LF, LG, LS, BX, BY, BZ>;
    using TC = typename C::TC;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *tile = reinterpret_cast<double *>(smem_raw);
    float2 *pops = reinterpret_cast<float2 *>(smem_raw + C::TILE_BYTES);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + C::TILE_BYTES + C::POPS_BYTES);
    constexpr int HX = BX / 2;
    const int t = threadIdx.x;
    const int tx = 2 * (t % HX), ty = (t / HX) % BY, tz = t / (HX * BY);
    const int x0 = blockIdx.x * BX;
    int y0, z0;
    tile_origin<3>(P, BY, BZ, y0, z0);
    const uint32_t bar_a = smem_u32(bar);
    if (t == 0) {
        mbar_init(bar_a, 1);
        fence_mbar_init();
        fence_proxy_async();
    }
    const int x = x0 + tx, y = y0 + ty, z = z0 + tz;
    const bool active = node_active<3>(P, x, y, z);   // nx is even: the second node of an active pair is active
    const bool bc = tile_touches_bc(P, x0, y0, z0, BX, BY, BZ);
    NodeGeom2 g;
    double2 po = make_double2(0.0, 0.0);
    if (active && !bc) {
        g = make_geom2(P, x, y, z);
        const SrcPairSmem<LF, LG, LS, C, Fields> src(P, Fd, g, tile, pops, bar_a, t, tx, ty, tz, po);
        src.prefetch();   // before the barrier below: the copies fly while the CTA assembles
        po = __ldg(reinterpret_cast<const double2 *>(
            Fd.phi_old + (((unsigned)(z + P.pz) * (unsigned)P.ppy + (unsigned)(y + 1)) * (unsigned)P.ppx + (unsigned)(x + P.xpad))));
    }
    if (t == 0) {
        pdl_wait();   // phi^{n+1} is K_phi's output, the only input the preceding launch writes
        mbar_expect_tx(bar_a, TC::BYTES);
        tma_load_3d(smem_u32(tile), &phi_map, bar_a, x0, y0, z0);
    }
    __syncthreads();   // the mbarrier is initialised before anybody waits on it
    if (!active) return;
    if (bc) {
#pragma unroll 1
        for (int k = 0; k < 2; ++k) {
            const NodeGeom g1 = make_geom(P, x + k, y, z);
            const SrcGlobalPhiSmem<LF, LG, LS, float, true, TC, Fields> src(P, Fd, g1, tile, bar_a, tx + k, ty, tz);
            node_update<LF, LG, LS, float, MODE>(P, Fd, g1, src);
        }
    } else {
        const SrcPairSmem<LF, LG, LS, C, Fields> src(P, Fd, g, tile, pops, bar_a, t, tx, ty, tz, po);
        node_update<LF, LG, LS, f2, MODE>(P2, Fd, g, src);
    }
}

// Tile of BX x BY x BZ NODES (the TMA box of the one-node kernel), BX / 2 x BY x BZ threads.
template <class LF, class LG, class LS, int MODE, int BX, int BY, int BZ, int MINB, class Fields>
__global__ void __launch_bounds__(BX / 2 * BY * BZ, MINB)
k_main_pair(const DevParams<float> P, const DevParams<f2> P2, const Fields Fd, const __grid_constant__ CUtensorMap phi_map) {
    using TC = PhiTileCfg<double, 3, BX, BY, BZ>;
    using SM = PhiTileSmem<double, TC>;
    __shared__ __align__(128) unsigned char smem_raw[SM::BYTES];
    double *tile = reinterpret_cast<double *>(smem_raw);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + SM::TILE_BYTES);
    constexpr int HX = BX / 2;
    const int t = threadIdx.x;
    const int tx = 2 * (t % HX), ty = (t / HX) % BY, tz = t / (HX * BY);
    const int x0 = blockIdx.x * BX;
    int y0, z0;
    tile_origin<3>(P, BY, BZ, y0, z0);
    const uint32_t bar_a = smem_u32(bar);
    if (t == 0) {
        mbar_init(bar_a, 1);
        fence_mbar_init();
        fence_proxy_async();
        pdl_wait();   // phi^{n+1} is K_phi's output: the only input of this kernel that the preceding launch writes
        mbar_expect_tx(bar_a, TC::BYTES);
        tma_load_3d(smem_u32(tile), &phi_map, bar_a, x0, y0, z0);
    }
    __syncthreads();   // the barrier is initialised before anybody waits on it
    const int x = x0 + tx, y = y0 + ty, z = z0 + tz;
    if (!node_active<3>(P, x, y, z)) return;   // nx is even: the second node of an active pair is active
    if (tile_touches_bc(P, x0, y0, z0, BX, BY, BZ)) {
#pragma unroll 1
        for (int k = 0; k < 2; ++k) {
            const NodeGeom g = make_geom(P, x + k, y, z);
            const SrcGlobalPhiSmem<LF, LG, LS, float, true, TC, Fields> src(P, Fd, g, tile, bar_a, tx + k, ty, tz);
            node_update<LF, LG, LS, float, MODE>(P, Fd, g, src);
        }
    } else {
        const NodeGeom2 g = make_geom2(P, x, y, z);
        const SrcPair<LF, LG, LS, TC, Fields> src(P, Fd, g, tile, bar_a, x, y, z, tx, ty, tz);
        node_update<LF, LG, LS, f2, MODE>(P2, Fd, g, src);
    }
}

}  // namespace lbm

namespace lbm {

// ---- K_phi for pairs (float populations, double phi, 3D): phi^{n+1} of the two nodes by the error-free sum of k_phi.cuh in packed
// arithmetic (the one-node kernel is issue-bound in float: 69% of the issue slots at 55% of the DRAM peak), 8-byte loads where the
// link does not move in x, one 16-byte store of the two doubles.  Nodes with ghost images and tiles on non-periodic faces take
// the one-node code.
__device__ __forceinline__ void two_sum2(f2 &hi, f2 &lo, f2 v) {   // Knuth: hi + lo + v = hi' + lo' exactly, both nodes at once
    const f2 s = add2(hi, v);
    const f2 bb = add2(s, -hi);
    lo = add2(lo, add2(add2(hi, -add2(s, -bb)), add2(v, -bb)));
    hi = s;
}

template <class LG, int BX, int BY, int BZ, int NPT>
__global__ void __launch_bounds__(BX / 2 * BY *BZ)
k_phi_pair(const DevParams<float> P, const float *__restrict__ g_in, double *__restrict__ phi_new) {
    pdl_launch_dependents();   // as k_phi
    constexpr int HX = BX / 2;
    const int t = threadIdx.x;
    const int x0 = blockIdx.x * BX, y0 = blockIdx.y * BY, z0 = P.s0 + blockIdx.z * BZ * NPT;   // this launch covers the layers [P.s0, P.s1)
    const int x = x0 + 2 * (t % HX), y = y0 + (t / HX) % BY, zb = z0 + t / (HX * BY);
    if (x >= P.nx || y >= P.ny) return;   // nx is even
    const unsigned N = (unsigned)P.N;
    if (tile_touches_bc(P, x0, y0, z0, BX, BY, BZ * NPT)) {
#pragma unroll 1
        for (int j = 0; j < 2 * NPT; ++j) {
            const int z = zb + (j >> 1) * BZ;
            if (z >= P.s1) break;
            const NodeGeom g = make_geom(P, x + (j & 1), y, z);
            float gi[LG::Q];
            pull<LG, float, true>(g_in, N, g, P.bc_g, P.bc_phi, gi);
            store_phi_with_images(phi_new, P, g, phi_sum<double>(gi));
        }
        return;
    }
    f2 gi[NPT][LG::Q];
    bool ok[NPT];
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        const int z = zb + j * BZ;
        ok[j] = z < P.s1;
        if (ok[j]) {
            const NodeGeom2 g = make_geom2(P, x, y, z);
            static_for<LG::Q>([&](auto ic) {
                constexpr int I = decltype(ic)::value;
                gi[j][I] = pull_pair<LG, I, false>(g_in, N, g);
            });
        }
    }
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        if (!ok[j]) continue;
        const int z = zb + j * BZ;
        f2 hi = gi[j][0], lo = f2(0.0f);
#pragma unroll
        for (int i = 1; i < LG::Q; ++i) two_sum2(hi, lo, gi[j][i]);
        const double v0 = (double)hi.x + (double)lo.x, v1 = (double)hi.y + (double)lo.y;
        const bool edge = y == 0 || y == P.ny - 1 || z == 0 || z == P.nz - 1;
        if (!edge) {   // at most the periodic images in x (store_phi_periodic_tile, k_phi.cuh)
            const long long pc = ((long long)(z + P.pz) * P.ppy + (y + 1)) * P.ppx + (x + P.xpad);
            *reinterpret_cast<double2 *>(phi_new + pc) = make_double2(v0, v1);   // x and xpad are even: 16-byte aligned
            if (x == 0) phi_new[pc + P.nx] = v0;
            if (x + 2 == P.nx) phi_new[pc + 1 - P.nx] = v1;
        } else {
            store_phi_with_images(phi_new, P, make_geom(P, x, y, z), v0);
            store_phi_with_images(phi_new, P, make_geom(P, x + 1, y, z), v1);
        }
    }
}

}  // namespace lbm
