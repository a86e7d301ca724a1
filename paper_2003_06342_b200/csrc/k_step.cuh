// The whole step (H1..H7) in ONE launch: K_phi and K_main work items interleaved along a sweep, so that what K_phi pulls and
// writes -- the Q_g populations of g and phi^{n+1} -- is read again by K_main a few megabytes of traffic later, out of L2
// instead of HBM: 70 instead of 78 values per lattice update in 3D, 51 instead of 61 in 2D.
//
// Work items (one CTA each, nothing persistent -- no loop-carried state to spill):
//   P item  K_phi on BX x 2 BM nodes of TWO consecutive layers of the slow axis (z in 3D, y in 2D), four nodes per thread:
//           phi^{n+1} = sum_i g_i (Eq.32) with its ghost images;
//   M item  K_main on one BX x BM tile of one layer (the tile bodies of k_main_smem.cuh / k_main_phitma.cuh).
// Order.  The mid axis (y in 3D) is cut into J blocks of By rows; block after block sweeps the slow axis in layer pairs:
// group k of a block holds the P items of pair position k and the M items of the pair that became computable `head`
// positions earlier.  P windows are shifted by one row against the M rows of a block (block 0 also takes the last row), so
// that every phi^{n+1} value an M item reads -- rows y-1..y+1, layers z-1..z+1, ghost images included -- belongs to a P
// item EARLIER in the order; nothing is computed twice.  The slow axis starts with its last pair for the same reason
// (periodic wrap).
// Hand-over.  P items wait for nobody.  A P CTA adds 1 to the counter of its (block, pair) slice with release semantics
// after its stores; an M CTA issues its asynchronous population copies first, then polls (acquire) the at most nine slice
// counters it depends on, then requests its phi box by TMA.  An item only ever waits for items earlier in the order; with
// `ticketed` the CTAs take their place in the order from a global ticket (atomicAdd), so those items are already running
// whatever the dispatch order of the hardware.  Counters run on monotonically over the launches.
#pragma once

#include "k_main_smem.cuh"
#include "k_phi.cuh"

namespace lbm {

struct StepItem {
    int role;               // 0 = P, 1 = M, 2 = empty slot
    int j, cls, pair;       // mid block, its class, layer pair
    int xi;                 // x tile
    int m0;                 // P: first entry of the block's row window; M: first row (mid axis) of the tile
    int layer;              // M: layer of the slow axis
};

// linear place L in the order -> work item (a handful of multiplications; every thread does it)
template <int BM> __device__ __forceinline__ StepItem decode_place(const SweepPlan &S, unsigned L) {
    StepItem it;
    const unsigned row = S.d_gx.div(L), bx = L - row * S.d_gx.d;     // L = (bz * gy + by) * gx + bx
    const unsigned bz = S.d_gy.div(row), by = row - bz * S.d_gy.d;
    it.j = (int)bz;
    it.cls = bz == 0 ? 0 : ((int)bz == S.J - 1 ? 2 : 1);
    if ((int)bx < S.cPmax) {
        // P order along the slow axis: the last pair first (its layers are the periodic neighbours of layer 0), then 0, 1, ...
        const int k = (int)by;
        it.pair = k == 0 ? S.NP - 1 : k - 1;
        const unsigned rt = S.d_xt.div(bx);
        it.xi = (int)(bx - rt * S.d_xt.d);
        it.m0 = (int)rt * 2 * BM;
        it.layer = 2 * it.pair;
        it.role = (k < S.NP && (int)rt < S.ptiles[it.cls]) ? 0 : 2;
    } else {
        unsigned r = bx - (unsigned)S.cPmax;
        const unsigned half = (unsigned)(S.mtmax * S.xt);
        const int q = r >= half ? 1 : 0;
        r -= q ? half : 0u;
        it.pair = (int)by - S.head;
        it.layer = 2 * it.pair + q;
        const unsigned rt = S.d_xt.div(r);
        it.xi = (int)(r - rt * S.d_xt.d);
        it.m0 = it.j * S.By + (int)rt * BM;
        it.role = (it.pair >= 0 && it.layer < S.nslow && (int)rt < S.mtiles[it.cls]) ? 1 : 2;
    }
    return it;
}

// row of the mid axis that entry k of block j's P window stands for
__device__ __forceinline__ int p_window_row(const SweepPlan &S, int j, int k) {
    if (S.J == 1) return k;
    if (j == 0) return k == 0 ? S.nmid - 1 : k - 1;
    return j * S.By + 1 + k;
}

// M item: the slices whose phi^{n+1} the tile reads.  Called by warp 0 before it issues anything else (so that the polls
// do not queue behind the tile's population copies); lanes 0..8 watch one counter each.  Gives up after about a second
// instead of hanging the device if the hand-over is ever broken.
struct WaitSlices {
    static constexpr bool WAITS = true;
    const SweepPlan &S;
    int j, layer;
    unsigned long long seen;   // thread 0: ticketed: epoch; else the count of CTAs that had arrived when this one did
    __device__ __forceinline__ void operator()() const {
        const int t = threadIdx.x;
        // launches completed before this one: all CTAs of a launch see the same value (k_step below)
        const unsigned long long v = __shfl_sync(0xffffffffu, seen, 0);
        if (t >= 9 || (S.xflags & 4)) return;
        const unsigned long long epoch = S.ticketed ? v : v / S.total;
        // layers layer-1, layer, layer+1 (wrapped: the periodic image of a layer is written by the item that owns it)
        const int d = t % 3 - 1;
        const int l = layer + d < 0 ? S.nslow - 1 : (layer + d >= S.nslow ? 0 : layer + d);
        const int pair = l >> 1;
        // blocks: own, the one before (rows j By - 1, j By), and block 0 for the last block (last row, image of row 0)
        const int which = t / 3;
        int jb;
        if (which == 0) jb = j;
        else if (which == 1) { if (j == 0) return; jb = j - 1; }
        else { if (j != S.J - 1 || S.J < 3) return; jb = 0; }
        const int cls = jb == 0 ? 0 : (jb == S.J - 1 ? 2 : 1);
        const unsigned long long target = (epoch + 1ull) * (unsigned long long)S.cP[cls];
        const unsigned long long *ctr = S.done + (size_t)jb * S.NP + pair;
        if (ld_acquire_gpu(ctr) >= target) return;
        const long long t0 = clock64();
        while (ld_acquire_gpu(ctr) < target) {
            __nanosleep(32);
            if (clock64() - t0 > (1ll << 31)) { *S.err = 1; return; }
        }
    }
};

// P item: K_phi on BX x 2 BM nodes (window entries m0 + tm and m0 + BM + tm) of the two layers of `pair`
template <class LG, class real, int BX, int BM, class sreal, class preal>
__device__ __forceinline__ void phi_item(const DevParams<real> &P, const SweepPlan &S, const StepItem &it,
                                         const sreal *__restrict__ g_in, preal *__restrict__ phi_new) {
    using vreal = typename std::conditional<std::is_same<real, sreal>::value, real, preal>::type;
    constexpr bool THREE_D = LG::D == 3;
    const int t = threadIdx.x;
    const int tx = t % BX, tm = t / BX;
    const int x = it.xi * BX + tx;
    const int l0 = it.layer;
    // does the item touch a non-periodic face?  (CTA-uniform)
    bool bc = false;
    {
        const unsigned m = P.bcfaces;
        const int xa = it.xi * BX;
        if (m & 3u) bc |= (xa == 0 && (m & 1u)) || (xa + BX >= P.nx && (m & 2u));
        const unsigned mmid = THREE_D ? (m >> 2) & 3u : 0u, mslow = THREE_D ? (m >> 4) & 3u : (m >> 2) & 3u;
        if (mmid) {
            for (int q = 0; q < 2 * BM; ++q) {
                if (it.m0 + q < S.prows[it.cls]) {
                    const int rq = p_window_row(S, it.j, it.m0 + q);
                    bc |= (rq == 0 && (mmid & 1u)) || (rq == S.nmid - 1 && (mmid & 2u));
                }
            }
        }
        if (mslow) bc |= (l0 == 0 && (mslow & 1u)) || (l0 + 2 >= S.nslow && (mslow & 2u));
    }
    vreal gi[4][LG::Q];
    NodeGeom g[4];
    bool ok[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int layer = l0 + (q & 1), k = it.m0 + (q >> 1) * BM + tm;
        ok[q] = x < P.nx && k < S.prows[it.cls] && layer < S.nslow;
        if (ok[q]) {
            const int row = p_window_row(S, it.j, k);
            g[q] = THREE_D ? make_geom(P, x, row, layer) : make_geom(P, x, layer, 0);
            if (bc) pull<LG, vreal, true>(g_in, (unsigned)P.N, g[q], P.bc_g, P.bc_phi, gi[q]);
            else pull<LG, vreal, false>(g_in, (unsigned)P.N, g[q], P.bc_g, P.bc_phi, gi[q]);
        }
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (ok[q]) store_phi_with_images(phi_new, P, g[q], phi_sum<preal>(gi[q]));
    }
    __syncthreads();   // every store of the CTA is ordered before the release below
    if (t == 0) red_release_gpu_add(S.done + (size_t)it.j * S.NP + it.pair, 1ull);
}

// POPS_SMEM: M items stage their populations in shared memory (k_main_smem.cuh), else gather into registers
template <class LF, class LG, class LS, class real, int MODE, int BX, int BM, int MINB, bool POPS_SMEM, bool STAGE_G, class Fields>
__global__ void __launch_bounds__(BX *BM, MINB)
k_step(const DevParams<real> P, const Fields Fd, typename Fields::preal *phi_new_w, const __grid_constant__ CUtensorMap phi_map,
       const SweepPlan S) {
    constexpr bool THREE_D = LF::D == 3;
    constexpr int BY = THREE_D ? BM : 1, BZ = 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned s_place;
    unsigned place;
    unsigned long long seen = 0;
    if (S.ticketed) {
        if (threadIdx.x == 0) {
            const unsigned long long tk = atomicAdd(S.ticket, 1ull);
            if ((unsigned)tk == S.total - 1u) atomicAdd(S.ticket, (1ull << 32) - (unsigned long long)S.total);   // next launch: epoch + 1, ticket 0
            s_place = (unsigned)tk;
            seen = tk >> 32;
        }
        __syncthreads();
        place = s_place;
    } else {
        place = blockIdx.x;
        // Launches completed so far = floor(left / total), the same for every CTA of a launch: `left` counts the CTAs of all
        // launches that have passed this point, each adds itself AFTER its own read, and a launch starts when the one before is over.
        if (threadIdx.x == 0) {
            seen = ld_relaxed_gpu(S.left);
            red_relaxed_gpu_add(S.left, 1ull);
        }
    }
    const StepItem it = decode_place<BM>(S, place);
    if (it.role == 0) phi_item<LG, real, BX, BM>(P, S, it, Fd.g_in, phi_new_w);
    else if (it.role == 1) {
        const int x0 = it.xi * BX, y0 = THREE_D ? it.m0 : it.layer, z0 = THREE_D ? it.layer : 0;
        const WaitSlices ready{S, it.j, it.layer, seen};
        if constexpr (POPS_SMEM) main_tile_smem<LF, LG, LS, real, MODE, BX, BY, BZ, STAGE_G>(P, Fd, &phi_map, smem_raw, x0, y0, z0, ready);
        else main_tile_phitma<LF, LG, LS, real, MODE, BX, BY, BZ>(P, Fd, &phi_map, smem_raw, x0, y0, z0, ready);
    }
}

}  // namespace lbm
