// Device code of the coupled phase-field LBM step (sm_100a).  Shares nothing with oracle/.
//
// Data layout in HBM:
//   populations  SoA [Q][z][y][x], two buffers per lattice (pull scheme, read A / write B, swap);
//   phi          padded [nz+2][ny+2][ppx] (2D: [ny+2][ppx]; node x at column x + xpad) with materialised ghost layers (periodic image,
//                zero-flux mirror, Dirichlet 2v - mirror), two buffers (level n and n+1);
//   Pdot, u, p, T  [z][y][x].
// Kernels:
//   k_phi   H1: pull g (+BC), phi^{n+1} = sum g + dt/2 Pdot (Eq.32; the Pdot term rides in the stored rest
//           population, k_main.cuh), ghost images.
//   k_main  H2..H7: stencils (Eq.35,36), closures, pull f,s,g (+BC), moments (Eq.28a,b, 34), production
//           refresh (Eq.18), BGK collision of the three lattices (Eq.25), store post-collision populations.
#pragma once

#include <cuda_runtime.h>
#include <type_traits>
#include <utility>

#include "lattices.cuh"

namespace lbm {

enum { BC_PERIODIC = 0, BC_BOUNCE = 1 /* wall / zero-flux */, BC_ANTI = 2 /* open / Dirichlet */ };
// MODE_STEP_PU: prescribed-velocity step (LBM_FLAG_PRESCRIBED_U): u is read from the macro array instead of Eq.(28a),
// p and T are stored every step.  A separate instantiation so that the production kernels carry no trace of it.
// MODE_STEP_VAR: step with one of the model variants of lbm_params.grad_scheme / div_scheme (biased directional derivatives,
// PAPER.md:318; stencil divergence of u phi, reading S17); stores u, p, T every step.  MODE_U: the velocity pass
// that precedes it when the divergence is a stencil (u^{n+1} of every node, Eq.28a, and nothing else).
// MODE_INIT_VAR: initialisation with a variant.
enum { MODE_STEP = 0, MODE_STEP_MACRO = 1, MODE_INIT = 2, MODE_STEP_PU = 3, MODE_STEP_VAR = 4, MODE_U = 5, MODE_INIT_VAR = 6 };
// modes that know the variants (all run the direct kernel; the production kernels and the plain initialisation carry no trace of them)
template <int MODE> struct mode_has_variants { static constexpr bool value = MODE == MODE_INIT_VAR || MODE == MODE_STEP_VAR || MODE == MODE_U; };
template <int MODE> struct mode_is_init { static constexpr bool value = MODE == MODE_INIT || MODE == MODE_INIT_VAR; };

// ---- compile-time loop over directions ---------------------------------------------------------------
template <class F, int... I>
__device__ __forceinline__ void static_for_impl(F &&f, std::integer_sequence<int, I...>) {
    (f(std::integral_constant<int, I>{}), ...);
}
template <int N, class F> __device__ __forceinline__ void static_for(F &&f) {
    static_for_impl(f, std::make_integer_sequence<int, N>{});
}

// e_i . v with e_i in {-1,0,1}^3 folded at compile time (no multiplications, no 0*x terms)
template <class L, int I, class real> __device__ __forceinline__ real dot_e(real v0, real v1, real v2) {
    real r = real(0);
    bool first = true;
    if constexpr (L::ex(I) != 0) { r = (L::ex(I) > 0) ? v0 : -v0; first = false; }
    if constexpr (L::ey(I) != 0) { r = first ? ((L::ey(I) > 0) ? v1 : -v1) : ((L::ey(I) > 0) ? r + v1 : r - v1); first = false; }
    if constexpr (L::ez(I) != 0) { r = first ? ((L::ez(I) > 0) ? v2 : -v2) : ((L::ez(I) > 0) ? r + v2 : r - v2); first = false; }
    (void)first;
    return r;
}

// ---- kernel parameters (passed by value) ------------------------------------------------------------------
template <class real> struct DevParams {
    int nx, ny, nz;
    int s0, s1;            // layers [s0, s1) of the slowest axis (z in 3D, y in 2D) that THIS launch of K_phi / K_main covers
    long long N;           // nx*ny*nz
    int ppx, ppy, pz;      // padded phi: row pitch, ny+2, z offset (1 in 3D, 0 in 2D)
    int xpad;              // padded phi: x offset of node 0 (16 bytes of elements, so TMA boxes start 16-byte aligned)
    long long pplane;      // ppx*ppy
    int bc_f[3][2], bc_g[3][2], bc_s[3][2];   // BC_* per face (f: wall->BOUNCE, open->ANTI)
    real bc_phi[3][2], bc_T[3][2], bc_p[3][2];
    int nonper[3];         // axis has non-periodic faces
    unsigned bcfaces;      // bit 2*axis + side: that face is non-periodic
    real dt, hdt, c, inv_dx, inv_dx2;
    real cs2f, cs2g, cs2s;           // e2 * c^2 per lattice
    real inv_cs2f, inv_cs2g, inv_cs2s;   // reciprocals, and c / cs2 per lattice (host-computed: no per-node divisions)
    real c_cs2f, c_cs2g, c_cs2s;
    real inv_dt, tauf_num, taus_den;     // 1/dt ; nu_l nu_g/(cs2f dt) ; 1/(cs2s dt)
    real rho_l, rho_g, rho_diff, drho;   // rho_g - rho_l ; 1/rho_g - 1/rho_l
    real nu_l, nu_g, nu_prod;            // nu_l * nu_g
    real fourH, K;                       // Eq.(14),(15b)
    real grav[3], force[3];
    real alpha_l, alpha_diff;            // alpha_g - alpha_l
    real M, om_g, cac;                   // mobility, 1/(M/(cs2g dt)+1/2), M*(4/W)/cs2g * c
    double g_om, g_dt, g_c_cs2, g_inv_cs2, g_cac;   // constants of the g collision, which runs in the phi type (k_main.cuh)
    real LCp, CpL, T_sat, theta_I, pc_coef;   // L/Cp, Cp/L, 4/(A W^2)
    real eps_n2;
    int phase_change, latent_heat, prescribed_u;
    int grad_scheme, div_scheme;   // LBM_GRAD_*, LBM_DIV_* (include/lbm.h)
};

// Storage types are separate from the arithmetic type `real` of the kernels (include/lbm.h "precision"):
//   sreal  populations, Pdot and the macro arrays (what streams through HBM every step);
//   preal  the padded phi arrays.  phi is kept in double even when everything else is float: dphi/dt =
//          (phi^{n+1} - phi^n)/dt (reading S4) is a difference of two O(1) numbers that enters T multiplied by L/Cp, so
//          the rounding of a float phi (6e-8) is the largest single error of an all-float step.
template <class sreal_, class preal_> struct DevFieldsT {
    using sreal = sreal_;
    using preal = preal_;
    const sreal *f_in, *g_in, *s_in;   // post-collision populations of the previous level
    sreal *f_out, *g_out, *s_out;      // post-collision populations of this level
    const preal *phi_new;              // padded, level n+1 (written by k_phi)
    const preal *phi_old;              // padded, level n
    const sreal *pdot_in;              // production field of level n (the stored one, reading S3)
    sreal *pdot;                       // production field of level n+1 (the array that belongs to the output buffers)
    sreal *u, *p, *T;                  // macro arrays: outputs (MODE_STEP_MACRO) or inputs (MODE_INIT)
};
template <class real> using DevFields = DevFieldsT<real, real>;   // one type throughout (fp64)

// ---- per-node geometry ------------------------------------------------------------------------------------
// Element offsets are 32-bit: Q * N < 2^32 is checked by the host (lbm_create).
struct NodeGeom {
    int x, y, z;
    unsigned n;           // own linear index
    unsigned sx[3];       // source x for e_x = -1, 0, +1  (x - e_x, wrapped)
    unsigned sy[3];       // source row offset (y - e_y wrapped) * nx
    unsigned sz[3];       // source plane offset (z - e_z wrapped) * nx*ny
    bool lo[3], hi[3];    // node sits on the first / last layer of the axis
};

template <class real>
__device__ __forceinline__ NodeGeom make_geom(const DevParams<real> &P, int x, int y, int z) {
    NodeGeom g;
    g.x = x; g.y = y; g.z = z;
    const unsigned row = (unsigned)P.nx, plane = (unsigned)P.nx * (unsigned)P.ny;
    g.n = (unsigned)z * plane + (unsigned)y * row + (unsigned)x;
    g.lo[0] = x == 0; g.hi[0] = x == P.nx - 1;
    g.lo[1] = y == 0; g.hi[1] = y == P.ny - 1;
    g.lo[2] = z == 0; g.hi[2] = z == P.nz - 1;
    g.sx[0] = g.hi[0] ? 0u : (unsigned)(x + 1);  g.sx[1] = (unsigned)x;  g.sx[2] = g.lo[0] ? (unsigned)(P.nx - 1) : (unsigned)(x - 1);
    g.sy[0] = (unsigned)(g.hi[1] ? 0 : y + 1) * row;  g.sy[1] = (unsigned)y * row;
    g.sy[2] = (unsigned)(g.lo[1] ? P.ny - 1 : y - 1) * row;
    g.sz[0] = (unsigned)(g.hi[2] ? 0 : z + 1) * plane;  g.sz[1] = (unsigned)z * plane;
    g.sz[2] = (unsigned)(g.lo[2] ? P.nz - 1 : z - 1) * plane;
    return g;
}

// element offset of the pull source of direction I (periodic wrap only)
template <class L, int I> __device__ __forceinline__ unsigned pull_offset(unsigned N, const NodeGeom &g) {
    return (unsigned)I * N + g.sz[L::ez(I) + 1] + g.sy[L::ey(I) + 1] + g.sx[L::ex(I) + 1];
}

// Loads.  ld_first: read-only path, free for the compiler to schedule.  ld_again: the SAME address read a second time
// (at collision time) -- opaque to common-subexpression elimination on purpose, so that the first value need not stay
// in a register for the whole step; it hits L1.
__device__ __forceinline__ double ld_again(const double *p) {
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld_again(const float *p) {
    float v;
    asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
template <bool AGAIN, class real, class sreal> __device__ __forceinline__ real ld_pop(const sreal *p) {
    if constexpr (AGAIN) return real(ld_again(p));
    else return real(__ldg(p));
}

// Pull-stream ONE direction of one lattice (theta* = theta(x + c_i dt, t + dt)).
// BC = false: every axis the node touches is periodic -> pure wrapped gather.
// BC = true : a link that leaves through a non-periodic face takes the post-collision opposite population of the
//             same node: bounce-back or anti-bounce-back -v + 2 w_i value;
//             tangential wrap first, lowest axis decides (reading S8).
// `real` is the type the value is returned (and the anti-bounce-back evaluated) in; the stored type and the type of the
// face values are deduced.
template <class L, int I, class real, bool BC, bool AGAIN = false, class sreal, class vreal>
__device__ __forceinline__ real pull_one(const sreal *__restrict__ src, unsigned N, const NodeGeom &g,
                                         const int (&bc)[3][2], const vreal (&val)[3][2]) {
    constexpr int ex = L::ex(I), ey = L::ey(I), ez = L::ez(I);
    const unsigned ns = (unsigned)I * N + g.sz[ez + 1] + g.sy[ey + 1] + g.sx[ex + 1];
    if constexpr (!BC || I == 0) {
        return ld_pop<AGAIN, real>(src + ns);
    } else {
        int kind = BC_PERIODIC;
        vreal v = vreal(0);
        if constexpr (ex != 0) {
            constexpr int side = ex > 0 ? 0 : 1;
            if ((side == 0 ? g.lo[0] : g.hi[0]) && bc[0][side] != BC_PERIODIC) { kind = bc[0][side]; v = val[0][side]; }
        }
        if constexpr (ey != 0) {
            constexpr int side = ey > 0 ? 0 : 1;
            if (kind == BC_PERIODIC && (side == 0 ? g.lo[1] : g.hi[1]) && bc[1][side] != BC_PERIODIC) { kind = bc[1][side]; v = val[1][side]; }
        }
        if constexpr (ez != 0) {
            constexpr int side = ez > 0 ? 0 : 1;
            if (kind == BC_PERIODIC && (side == 0 ? g.lo[2] : g.hi[2]) && bc[2][side] != BC_PERIODIC) { kind = bc[2][side]; v = val[2][side]; }
        }
        if (kind == BC_PERIODIC) return ld_pop<AGAIN, real>(src + ns);
        const real back = ld_pop<AGAIN, real>(src + (unsigned)L::opp(I) * N + g.n);
        return kind == BC_BOUNCE ? back : real(2.0 * L::w(I)) * real(v) - back;
    }
}

template <class L, class real, bool BC, class sreal, class vreal>
__device__ __forceinline__ void pull(const sreal *__restrict__ src, unsigned N, const NodeGeom &g,
                                     const int (&bc)[3][2], const vreal (&val)[3][2], real (&out)[L::Q]) {
    static_for<L::Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        out[I] = pull_one<L, I, real, BC>(src, N, g, bc, val);
    });
}

// A position up to two layers outside the grid -> the node whose value stands for it: through a periodic face the periodic
// image, through any other face the mirror image in the face, which sits half a cell outside the first / last node
// (-1 -> 0, -2 -> 1).  cross[a] = 0, or 1 + side of the non-periodic face crossed on axis a (the caller applies that face's
// rule to the value).  Used by the variant modes only (second neighbours of the biased difference, neighbour velocities).
template <class real>
__device__ __forceinline__ void ghost_source(const DevParams<real> &P, const int (&bc)[3][2], int (&q)[3], int (&cross)[3]) {
    const int len[3] = {P.nx, P.ny, P.nz};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        cross[a] = 0;
        if (q[a] < 0) {
            if (bc[a][0] == BC_PERIODIC) q[a] += len[a];
            else { q[a] = -1 - q[a]; cross[a] = 1; }
        } else if (q[a] >= len[a]) {
            if (bc[a][1] == BC_PERIODIC) q[a] -= len[a];
            else { q[a] = 2 * len[a] - 1 - q[a]; cross[a] = 2; }
        }
    }
}

// Origin of a CTA's tile and activity of a node for launches that cover the layers [P.s0, P.s1) of the slowest axis
// (whole grid: 0 .. nz, or 0 .. ny in 2D; slab contexts launch their boundary layers and their interior separately).
template <int D, class real>
__device__ __forceinline__ void tile_origin(const DevParams<real> &P, int BY, int BZ, int &y0, int &z0) {
    if (D == 3) { y0 = blockIdx.y * BY; z0 = P.s0 + blockIdx.z * BZ; }
    else { y0 = P.s0 + blockIdx.y * BY; z0 = 0; }
}
template <int D, class real> __device__ __forceinline__ bool node_active(const DevParams<real> &P, int x, int y, int z) {
    return D == 3 ? (x < P.nx && y < P.ny && z < P.s1) : (x < P.nx && y < P.s1);
}

// does the tile [x0,x0+bx) x [y0,y0+by) x [z0,z0+bz) touch a non-periodic face?  (block-uniform)
template <class real>
__device__ __forceinline__ bool tile_touches_bc(const DevParams<real> &P, int x0, int y0, int z0, int bx, int by, int bz) {
    bool t = false;
    // per face (bit 2*axis + side of P.bcfaces): the ghost side of a slab is periodic-kind although the other end of the
    // axis is a physical face
    const unsigned m = P.bcfaces;
    if (m & 3u) t |= (x0 == 0 && (m & 1u)) || (x0 + bx >= P.nx && (m & 2u));
    if (m & 12u) t |= (y0 == 0 && (m & 4u)) || (y0 + by >= P.ny && (m & 8u));
    if (m & 48u) t |= (z0 == 0 && (m & 16u)) || (z0 + bz >= P.nz && (m & 32u));
    return t;
}

}  // namespace lbm
