// K_fused (3D): the whole step H1..H7 in ONE kernel -- no K_phi, no phi^{n+1} hand-off through HBM.
//
// A CTA owns a column of BX x BY nodes and marches LZ planes in z.  For every plane it needs it first computes
// phi^{n+1} = sum_i g*_i(x - e_i) [+BC]  (Eq.32; its dt/2 Pdot^n rides in the stored g*_0, k_main.cuh) on the plane INCLUDING a one-cell halo in
// x and y, straight from the post-collision g* of the previous level, into a ring of four shared-memory planes
// (z-1, z, z+1 in use, z+2 being filled).  The halo values are recomputed by the neighbouring CTAs as well: identical
// arithmetic, identical bits, served by L2 -- the price for dropping K_phi's 9 values per node of HBM traffic
// (step: 78 -> 70 values per lattice update).  Ghost values outside non-periodic faces are the mirror / Dirichlet images of
// DESIGN.md S8.
#pragma once

#include <cstdint>

#include "k_main.cuh"

namespace lbm {

// phi^{n+1} at a position that may lie one cell outside the domain: value at the wrapped / mirrored source node,
// Dirichlet transforms composed in axis order x, y, z (same definition as store_phi_with_images in k_phi.cuh).
template <class LG, class real, bool BC>
__device__ __forceinline__ real phi_new_at(const DevParams<real> &P, const real *__restrict__ g_in,
                                           const real *__restrict__ pdot_in, int x, int y, int z) {
    int q[3] = {x, y, z};
    const int len[3] = {P.nx, P.ny, P.nz};
    int kind[3] = {BC_PERIODIC, BC_PERIODIC, BC_PERIODIC};
    real val[3] = {real(0), real(0), real(0)};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (q[a] < 0 || q[a] >= len[a]) {
            const int side = q[a] < 0 ? 0 : 1;
            if (!BC || P.bc_g[a][side] == BC_PERIODIC) {
                q[a] += q[a] < 0 ? len[a] : -len[a];
            } else {
                q[a] = side == 0 ? 0 : len[a] - 1;
                kind[a] = P.bc_g[a][side];
                val[a] = P.bc_phi[a][side];
            }
        }
    }
    const NodeGeom g = make_geom(P, q[0], q[1], q[2]);
    real gi[LG::Q];
    pull<LG, real, BC>(g_in, (unsigned)P.N, g, P.bc_g, P.bc_phi, gi);
    real v = gi[0];
#pragma unroll
    for (int i = 1; i < LG::Q; ++i) v += gi[i];
    if constexpr (BC) {
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (kind[a] == BC_ANTI) v = real(2) * val[a] - v;
    }
    return v;
}

// cp.async (LDGSTS): global -> shared without staging registers; 8-byte (fp64) or 4-byte (fp32) elements
__device__ __forceinline__ void cp_async_elem(double *dst_smem, const double *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_elem(float *dst_smem, const float *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <class LF, class LG, class LS, class real, bool BC, int PX, int PY> struct SrcFused {
    const DevParams<real> &P;
    const DevFields<real> &Fd;
    const NodeGeom &g;
    const real *ring;     // 4 planes of PX * PY
    int slot;             // ring slot of the node's own plane
    int off;              // (ty + 1) * PX + tx + 1
    unsigned pcoff;
    __device__ __forceinline__ SrcFused(const DevParams<real> &P_, const DevFields<real> &Fd_, const NodeGeom &g_,
                                        const real *ring_, int slot_, int tx, int ty)
        : P(P_), Fd(Fd_), g(g_), ring(ring_), slot(slot_), off((ty + 1) * PX + tx + 1) {
        pcoff = ((unsigned)(g.z + P.pz) * (unsigned)P.ppy + (unsigned)(g.y + 1)) * (unsigned)P.ppx + (unsigned)(g.x + P.xpad);
    }
    __device__ __forceinline__ void pops_ready() const {}
    __device__ __forceinline__ void f_ready() const {}
    __device__ __forceinline__ void phi_ready() const {}
    __device__ __forceinline__ real phi(int dx, int dy, int dz) const {
        return ring[((slot + dz) & 3) * (PX * PY) + off + dx + dy * PX];
    }
    __device__ __forceinline__ real phi_old() const { return __ldg(Fd.phi_old + pcoff); }
    __device__ __forceinline__ real pdot_old() const { return __ldg(Fd.pdot_in + g.n); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real f() const { return pull_one<LF, I, real, BC, AGAIN>(Fd.f_in, (unsigned)P.N, g, P.bc_f, P.bc_p); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real s() const { return pull_one<LS, I, real, BC, AGAIN>(Fd.s_in, (unsigned)P.N, g, P.bc_s, P.bc_T); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real gg() const { return pull_one<LG, I, real, BC, AGAIN>(Fd.g_in, (unsigned)P.N, g, P.bc_g, P.bc_phi); }
};

template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int LZ, int MINB>
__global__ void __launch_bounds__(BX *BY, MINB)
k_main_fused(const DevParams<real> P, const DevFields<real> Fd, real *__restrict__ phi_out) {
    constexpr int PX = BX + 2, PY = BY + 2, NE = PX * PY, NT = BX * BY;
    __shared__ real ring[4 * NE];
    const int t = threadIdx.x;
    const int tx = t % BX, ty = t / BX;
    const int x0 = blockIdx.x * BX, y0 = blockIdx.y * BY, z0 = blockIdx.z * LZ;
    const int x = x0 + tx, y = y0 + ty;
    const int zend = min(z0 + LZ, P.nz);
    // x / y part of "this plane needs boundary rules": the tile grown by its halo touches a non-periodic face
    const bool bc_xy_phi = (P.nonper[0] && (x0 <= 1 || x0 + BX >= P.nx - 1)) || (P.nonper[1] && (y0 <= 1 || y0 + BY >= P.ny - 1));
    const bool bc_xy_node = (P.nonper[0] && (x0 == 0 || x0 + BX >= P.nx)) || (P.nonper[1] && (y0 == 0 || y0 + BY >= P.ny));

    // fill one phi^{n+1} plane (with halo) into its ring slot
    auto fill_plane = [&](int z) {
        real *dst = ring + (z & 3) * NE;      // z >= -1: (-1 & 3) == 3, consistent with (slot + dz) & 3
        const bool bc = bc_xy_phi || (P.nonper[2] && (z <= 0 || z >= P.nz - 1));
        for (int e = t; e < NE; e += NT) {
            const int ex = x0 - 1 + e % PX, ey = y0 - 1 + e / PX;
            real v = real(0);
            if (ex <= P.nx && ey <= P.ny)     // entries beyond the ragged edge + halo are never read
                v = bc ? phi_new_at<LG, real, true>(P, Fd.g_in, Fd.pdot_in, ex, ey, z)
                       : phi_new_at<LG, real, false>(P, Fd.g_in, Fd.pdot_in, ex, ey, z);
            dst[e] = v;
        }
    };

    // Asynchronous form of fill_plane for planes that need no boundary rule: issue() starts the copies of the LG::Q
    // pulled g* values of every entry this thread owns into stage[k][e]; reduce() sums them in the same
    // order as phi_new_at (so both forms give the same bits) once the copies have landed.
    constexpr int NEP = (NE + 31) / 32 * 32;
    __shared__ real stage[LG::Q * NEP];
    auto plane_is_plain = [&](int z) { return !(bc_xy_phi || (P.nonper[2] && (z <= 0 || z >= P.nz - 1))); };
    auto issue = [&](int z) {
        for (int e = t; e < NE; e += NT) {
            int ex = x0 - 1 + e % PX, ey = y0 - 1 + e / PX, ez = z;
            if (ex <= P.nx && ey <= P.ny) {
                ex += ex < 0 ? P.nx : (ex >= P.nx ? -P.nx : 0);
                ey += ey < 0 ? P.ny : (ey >= P.ny ? -P.ny : 0);
                ez += ez < 0 ? P.nz : (ez >= P.nz ? -P.nz : 0);
                const NodeGeom g = make_geom(P, ex, ey, ez);
                static_for<LG::Q>([&](auto ic) {
                    constexpr int I = decltype(ic)::value;
                    cp_async_elem(&stage[I * NEP + e],
                                  Fd.g_in + ((unsigned)I * (unsigned)P.N + g.sz[LG::ez(I) + 1] + g.sy[LG::ey(I) + 1] + g.sx[LG::ex(I) + 1]));
                });
            }
        }
        cp_async_commit();
    };
    auto reduce = [&](int z) {
        real *dst = ring + (z & 3) * NE;
        for (int e = t; e < NE; e += NT) {
            const int ex = x0 - 1 + e % PX, ey = y0 - 1 + e / PX;
            real v = real(0);
            if (ex <= P.nx && ey <= P.ny) {
                v = stage[e];
#pragma unroll
                for (int i = 1; i < LG::Q; ++i) v += stage[i * NEP + e];
            }
            dst[e] = v;
        }
    };

    fill_plane(z0 - 1);
    fill_plane(z0);
    bool pending = false;
    if (plane_is_plain(z0 + 1)) { issue(z0 + 1); pending = true; }
    for (int z = z0; z < zend; ++z) {
        if (pending) { cp_async_wait_all(); reduce(z + 1); }
        else fill_plane(z + 1);
        __syncthreads();                       // planes z-1, z, z+1 complete; plane z-2's slot is free for z+2
        pending = false;
        if (z + 1 < zend && plane_is_plain(z + 2)) { issue(z + 2); pending = true; }   // overlaps node_update(z)
        if (x < P.nx && y < P.ny) {
            const NodeGeom g = make_geom(P, x, y, z);
            const real phi_c = ring[(z & 3) * NE + (ty + 1) * PX + tx + 1];
            phi_out[((unsigned)(z + P.pz) * (unsigned)P.ppy + (unsigned)(y + 1)) * (unsigned)P.ppx + (unsigned)(x + P.xpad)] = phi_c;
            if (bc_xy_node || (P.nonper[2] && (z == 0 || z == P.nz - 1))) {
                const SrcFused<LF, LG, LS, real, true, PX, PY> src(P, Fd, g, ring, z & 3, tx, ty);
                node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
            } else {
                const SrcFused<LF, LG, LS, real, false, PX, PY> src(P, Fd, g, ring, z & 3, tx, ty);
                node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
            }
        }
    }
}

}  // namespace lbm
