// K_phi (step H1): phi^{n+1} = sum_i g_i + dt/2 sum_i P_i^g  (Eq.32) from the pulled, boundary-treated
// g populations, written into the padded phi array together with its ghost images so that K_main's stencils
// (and its TMA halo boxes) never leave the array.
#pragma once

#include "kernels.cuh"
#include "ptx.cuh"

namespace lbm {

// Store phi of node g into the padded array and into every ghost image of that node (reading S8-iv):
// periodic axis -> image one period away; zero-flux face -> mirror phi(-1) = phi(0); Dirichlet face with value v ->
// phi(-1) = 2 v - phi(0).  Transforms compose in axis order x, y, z (what an axis-by-axis ghost fill would give).
template <class real, class preal>
__device__ __forceinline__ void store_phi_with_images(preal *__restrict__ phi_pad, const DevParams<real> &P,
                                                      const NodeGeom &g, preal v) {
    const long long pc = ((long long)(g.z + P.pz) * P.ppy + (g.y + 1)) * P.ppx + (g.x + P.xpad);
    phi_pad[pc] = v;
    const bool edge = g.lo[0] | g.hi[0] | g.lo[1] | g.hi[1] | (P.pz && (g.lo[2] | g.hi[2]));
    if (!edge) return;
    int cnt[3];
    long long off[3][3];
    int kind[3][3];
    real bval[3][3];
    const long long stride[3] = {1, P.ppx, P.pplane};
    const int len[3] = {P.nx, P.ny, P.nz};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        cnt[a] = 1; off[a][0] = 0; kind[a][0] = BC_PERIODIC; bval[a][0] = real(0);
        if (a == 2 && !P.pz) continue;
        // A periodic-kind face opposite a non-periodic one is the ghost side of a slab (include/lbm.h, halo): its layer has
        // no image -- the pad layer one period away belongs to the physical face there.
        const bool both_per = P.bc_g[a][0] == BC_PERIODIC && P.bc_g[a][1] == BC_PERIODIC;
        if (g.lo[a]) {
            if (P.bc_g[a][0] == BC_PERIODIC) {
                if (both_per) { const int k = cnt[a]++; off[a][k] = (long long)len[a] * stride[a]; kind[a][k] = BC_PERIODIC; bval[a][k] = real(0); }
            } else { const int k = cnt[a]++; off[a][k] = -stride[a]; kind[a][k] = P.bc_g[a][0]; bval[a][k] = P.bc_phi[a][0]; }
        }
        if (g.hi[a]) {
            if (P.bc_g[a][1] == BC_PERIODIC) {
                if (both_per) { const int k = cnt[a]++; off[a][k] = -(long long)len[a] * stride[a]; kind[a][k] = BC_PERIODIC; bval[a][k] = real(0); }
            } else { const int k = cnt[a]++; off[a][k] = stride[a]; kind[a][k] = P.bc_g[a][1]; bval[a][k] = P.bc_phi[a][1]; }
        }
    }
    for (int i2 = 0; i2 < cnt[2]; ++i2)
        for (int i1 = 0; i1 < cnt[1]; ++i1)
            for (int i0 = 0; i0 < cnt[0]; ++i0) {
                if ((i0 | i1 | i2) == 0) continue;
                preal w = v;
                if (kind[0][i0] == BC_ANTI) w = preal(2) * preal(bval[0][i0]) - w;
                if (kind[1][i1] == BC_ANTI) w = preal(2) * preal(bval[1][i1]) - w;
                if (kind[2][i2] == BC_ANTI) w = preal(2) * preal(bval[2][i2]) - w;
                phi_pad[pc + off[0][i0] + off[1][i1] + off[2][i2]] = w;
            }
}

// Store phi of a node of a tile that touches NO non-periodic face.  Such a node can only have periodic images; the common one --
// the node sits on the first or last column of a periodic row and nowhere else on the edge of the grid -- is ONE extra store, one
// period away in x.  (Every row has two such nodes, so a quarter of the warps of a 256-wide grid would otherwise walk through
// the general image tables of store_phi_with_images for the sake of one lane.)  Rows and planes on the edge take the general path.
template <class real, class preal>
__device__ __forceinline__ void store_phi_periodic_tile(preal *__restrict__ phi_pad, const DevParams<real> &P, const NodeGeom &g, preal v) {
    if (g.lo[1] | g.hi[1] | (P.pz && (g.lo[2] | g.hi[2]))) { store_phi_with_images(phi_pad, P, g, v); return; }
    const long long pc = ((long long)(g.z + P.pz) * P.ppy + (g.y + 1)) * P.ppx + (g.x + P.xpad);
    phi_pad[pc] = v;
    if (g.lo[0]) phi_pad[pc + P.nx] = v;
    if (g.hi[0]) phi_pad[pc - P.nx] = v;
}

// Each thread handles NPT nodes, NPT tiles apart along the slowest tiled axis (z in 3D, y in 2D); all 8 NPT loads are
// issued before the first sum, which is what a latency-bound streaming kernel needs (measured: DESIGN.md "Kernels").
// phi^{n+1} = sum_i g_i + dt/2 Pdot (Eq.32); the last term is already inside the stored rest population (k_main.cuh), so
// this is a plain sum of the pulled values, in the type of the phi array (preal), so that with float populations and a double phi
// the result carries only the storage rounding of the populations.  Plain sum when the values already are preal;
// when an all-float kernel feeds a double phi the sum is an error-free float accumulation (Knuth two-sum: hi + lo is the
// exact sum) widened once at the end -- two conversions per node instead of Q_g + 1 (F2F.F64.F32 issues at a fraction
// of the FADD rate; K_phi on config 4 in fp32: 0.479 ms with the conversions, 0.306 ms with the two-sum).
__device__ __forceinline__ void two_sum(float &hi, float &lo, float v) {
    const float s = __fadd_rn(hi, v);
    const float bb = __fsub_rn(s, hi);
    lo = __fadd_rn(lo, __fadd_rn(__fsub_rn(hi, __fsub_rn(s, bb)), __fsub_rn(v, bb)));
    hi = s;
}
template <class preal, class vreal, int Q>
__device__ __forceinline__ preal phi_sum(const vreal (&gi)[Q]) {
    if constexpr (std::is_same<vreal, float>::value && std::is_same<preal, double>::value) {
        float hi = gi[0], lo = 0.0f;
#pragma unroll
        for (int i = 1; i < Q; ++i) two_sum(hi, lo, gi[i]);
        return (double)hi + (double)lo;
    } else {
        preal sum = preal(gi[0]);
#pragma unroll
        for (int i = 1; i < Q; ++i) sum += preal(gi[i]);
        return sum;
    }
}

// Each thread handles NPT nodes, NPT tiles apart along the slowest tiled axis (z in 3D, y in 2D); all 8 NPT loads are
// issued before the first sum, which is what a latency-bound streaming kernel needs (measured: DESIGN.md "Kernels").
// The pulled values are held in the arithmetic type `real` when that is the stored type (all-float kernels: no widening
// before the error-free sum), else in preal.
template <class LG, class real, int BX, int BY, int BZ, int NPT, class sreal, class preal>
__global__ void __launch_bounds__(BX *BY *BZ)
k_phi(const DevParams<real> P, const sreal *__restrict__ g_in, preal *__restrict__ phi_new) {
    using vreal = typename std::conditional<std::is_same<real, sreal>::value, real, preal>::type;
    constexpr bool ALONG_Z = LG::D == 3;
    pdl_launch_dependents();   // K_main may start filling the SMs as this grid drains; it waits (griddepcontrol.wait) before it reads phi
    const int t = threadIdx.x;
    const int x0 = blockIdx.x * BX;
    const int y0 = ALONG_Z ? blockIdx.y * BY : P.s0 + blockIdx.y * BY * NPT;   // this launch covers the layers [P.s0, P.s1)
    const int z0 = ALONG_Z ? P.s0 + blockIdx.z * BZ * NPT : 0;
    const int x = x0 + t % BX, yb = y0 + (t / BX) % BY, zb = z0 + t / (BX * BY);
    if (x >= P.nx) return;
    const bool bc = tile_touches_bc(P, x0, y0, z0, BX, BY * (ALONG_Z ? 1 : NPT), BZ * (ALONG_Z ? NPT : 1));
    vreal gi[NPT][LG::Q];
    NodeGeom g[NPT];
    bool ok[NPT];
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        const int y = yb + (ALONG_Z ? 0 : j * BY), z = zb + (ALONG_Z ? j * BZ : 0);
        ok[j] = ALONG_Z ? (y < P.ny && z < P.s1) : (y < P.s1);
        if (ok[j]) {
            g[j] = make_geom(P, x, y, z);
            if (bc) pull<LG, vreal, true>(g_in, (unsigned)P.N, g[j], P.bc_g, P.bc_phi, gi[j]);
            else pull<LG, vreal, false>(g_in, (unsigned)P.N, g[j], P.bc_g, P.bc_phi, gi[j]);
        }
    }
#pragma unroll
    for (int j = 0; j < NPT; ++j) {
        if (!ok[j]) continue;
        if (bc) store_phi_with_images(phi_new, P, g[j], phi_sum<preal>(gi[j]));
        else store_phi_periodic_tile(phi_new, P, g[j], phi_sum<preal>(gi[j]));
    }
}

// Initialisation helper: copy a plain [z][y][x] phi into both padded buffers with ghost images.
template <class real, int BX, int BY, int BZ, class sreal, class preal>
__global__ void __launch_bounds__(BX *BY *BZ)
k_phi_fill(const DevParams<real> P, const sreal *__restrict__ phi_plain, preal *__restrict__ pad_a, preal *__restrict__ pad_b) {
    const int t = threadIdx.x;
    const int x = blockIdx.x * BX + t % BX, y = blockIdx.y * BY + (t / BX) % BY, z = blockIdx.z * BZ + t / (BX * BY);
    if (x >= P.nx || y >= P.ny || z >= P.nz) return;
    const NodeGeom g = make_geom(P, x, y, z);
    const preal v = preal(phi_plain[g.n]);
    store_phi_with_images(pad_a, P, g, v);
    store_phi_with_images(pad_b, P, g, v);
}

// Debug / parity: streamed (post-pull, post-BC) populations of one lattice, all directions, to a [Q][N] scratch.
// `pdot_fold` (g only, else null): the production field folded into the stored rest population of `src` (k_main.cuh), taken out
// again so that the caller sees the populations of the paper.
template <class L, class real, int BX, int BY, int BZ, class sreal>
__global__ void __launch_bounds__(BX *BY *BZ)
k_stream_only(const DevParams<real> P, const sreal *__restrict__ src, sreal *__restrict__ dst, int which,
              const sreal *__restrict__ pdot_fold) {
    const int t = threadIdx.x;
    const int x = blockIdx.x * BX + t % BX, y = blockIdx.y * BY + (t / BX) % BY, z = blockIdx.z * BZ + t / (BX * BY);
    if (x >= P.nx || y >= P.ny || z >= P.nz) return;
    const NodeGeom g = make_geom(P, x, y, z);
    real v[L::Q];
    if (which == 0) pull<L, real, true>(src, (unsigned)P.N, g, P.bc_f, P.bc_p, v);
    else if (which == 1) pull<L, real, true>(src, (unsigned)P.N, g, P.bc_g, P.bc_phi, v);
    else pull<L, real, true>(src, (unsigned)P.N, g, P.bc_s, P.bc_T, v);
    if (pdot_fold) v[0] -= P.hdt * real(pdot_fold[g.n]);
#pragma unroll
    for (int i = 0; i < L::Q; ++i) dst[(size_t)i * P.N + g.n] = sreal(v[i]);
}

// Debug / parity: the stored rest population of g without the folded dt/2 Pdot (k_main.cuh).
template <class real, class sreal> __global__ void k_unfold_g0(sreal *__restrict__ dst, const sreal *__restrict__ g0,
                                                              const sreal *__restrict__ pdot, long long n, real hdt) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = sreal(real(g0[i]) - hdt * real(pdot[i]));
}

template <class real> __global__ void k_fill(real *__restrict__ dst, long long n, real v) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = v;
}

// unpadded copy of phi (for lbm_read_macro)
template <class real, int BX, int BY, int BZ, class sreal, class preal>
__global__ void __launch_bounds__(BX *BY *BZ)
k_phi_unpad(const DevParams<real> P, const preal *__restrict__ pad, sreal *__restrict__ plain) {
    const int t = threadIdx.x;
    const int x = blockIdx.x * BX + t % BX, y = blockIdx.y * BY + (t / BX) % BY, z = blockIdx.z * BZ + t / (BX * BY);
    if (x >= P.nx || y >= P.ny || z >= P.nz) return;
    plain[(long long)z * P.nx * P.ny + (long long)y * P.nx + x] =
        sreal(pad[((long long)(z + P.pz) * P.ppy + (y + 1)) * P.ppx + (x + P.xpad)]);
}

}  // namespace lbm
