// K_main (steps H2..H7): one thread per lattice node, everything between the pull and the post-collision store in
// registers.  Citations are PAPER.md:<line>; readings (G*/S*) are listed in DESIGN.md.
#pragma once

#include "kernels.cuh"

namespace lbm {

__device__ __forceinline__ double rsqrt_(double a) { return rsqrt(a); }
__device__ __forceinline__ float rsqrt_(float a) { return rsqrtf(a); }

// phi^{n+1} neighbourhood straight from the padded global array (L1/L2 serve the 18 re-reads)
template <class real> struct PhiGlobal {
    const real *__restrict__ c;   // pointer to the node's own padded element
    long long sy, sz;             // row pitch, plane pitch
    __device__ __forceinline__ real operator()(int dx, int dy, int dz) const { return __ldg(c + dx + dy * sy + dz * sz); }
};

// phi^{n+1} neighbourhood from a shared-memory halo tile (filled by TMA)
template <class real> struct PhiShared {
    const real *c;                // pointer to the node's own element in the tile
    int sy, sz;
    __device__ __forceinline__ real operator()(int dx, int dy, int dz) const { return c[dx + dy * sy + dz * sz]; }
};

template <class LF, class LG, class LS, class real, int MODE, bool BC, class PhiAcc>
__device__ __forceinline__ void node_update(const DevParams<real> &P, const DevFields<real> &Fd, const NodeGeom &g,
                                            const PhiAcc &ph) {
    const long long n = g.n;
    const long long N = P.N;

    // ---- H2: grad phi, lap phi by directional derivatives on the NS lattice (Eq.35a,b 36a,b; PAPER.md:291-315;
    //      the printed factor 3 is 1/e2, reading S2).  Opposite directions are paired: one difference, one sum.
    const real phi = ph(0, 0, 0);
    real gx = real(0), gy = real(0), gz = real(0), lsum = real(0);
    static_for<LF::Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        if constexpr (I > 0 && I < LF::opp(I)) {
            constexpr int ex = LF::ex(I), ey = LF::ey(I), ez = LF::ez(I);
            const real pp = ph(ex, ey, ez), pm = ph(-ex, -ey, -ez);
            const real d = pp - pm;
            constexpr real w = real(LF::w(I));
            if constexpr (ex != 0) gx += (ex > 0 ? w : -w) * d;
            if constexpr (ey != 0) gy += (ey > 0 ? w : -w) * d;
            if constexpr (ez != 0) gz += (ez > 0 ? w : -w) * d;
            lsum += w * (pp + pm);
        }
    });
    {
        const real sg = P.inv_dx * real(1.0 / LF::e2);
        gx *= sg; gy *= sg; gz *= sg;
    }
    const real lap = real(2.0 / LF::e2) * P.inv_dx2 * (lsum - real(1.0 - LF::w(0)) * phi);

    // ---- H3: local closures
    const real rho = P.rho_l + phi * P.rho_diff;                               // Eq.(1a)
    const real mu = P.fourH * phi * (phi - real(1)) * (phi - real(0.5)) - P.K * lap;   // Eq.(14)
    const real bu = rho - P.rho_l;                                             // buoyancy factor, reading G6
    const real Fx = mu * gx + bu * P.grav[0];                                  // Eq.(12),(13) PAPER.md:106-114
    const real Fy = mu * gy + bu * P.grav[1];
    const real Fz = mu * gz + bu * P.grav[2];
    const real grx = P.rho_diff * gx, gry = P.rho_diff * gy, grz = P.rho_diff * gz;   // grad rho
    const real alpha = P.alpha_l + phi * P.alpha_diff;                         // reading S6

    real ux, uy, uz, p, T, dtphi;
    real f[LF::Q], s[LS::Q];
    if constexpr (MODE == MODE_INIT) {
#pragma unroll
        for (int i = 0; i < LF::Q; ++i) f[i] = real(0);   // unused in this mode (bar = eq - dt/2 S)
#pragma unroll
        for (int i = 0; i < LS::Q; ++i) s[i] = real(0);
        ux = Fd.u[n]; uy = Fd.u[N + n]; uz = (LF::D == 3) ? Fd.u[2 * N + n] : real(0);
        p = Fd.p[n]; T = Fd.T[n]; dtphi = real(0);
    } else {
        // ---- H4: NS moments (Eq.28a)
        pull<LF, real, BC>(Fd.f_in, N, g, P.bc_f, P.bc_p, f);
        real m0 = real(0), mx = real(0), my = real(0), mz = real(0);
        static_for<LF::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            m0 += f[I];
            if constexpr (LF::ex(I) != 0) mx += LF::ex(I) > 0 ? f[I] : -f[I];
            if constexpr (LF::ey(I) != 0) my += LF::ey(I) > 0 ? f[I] : -f[I];
            if constexpr (LF::ez(I) != 0) mz += LF::ez(I) > 0 ? f[I] : -f[I];
        });
        const real inv_rho = real(1) / rho;
        const real cm = P.c / P.cs2f;
        ux = (cm * mx + P.hdt * Fx) * inv_rho;
        uy = (cm * my + P.hdt * Fy) * inv_rho;
        uz = (cm * mz + P.hdt * Fz) * inv_rho;
        // ---- H1 (time derivative), H5: heat moment with the STORED production rate (reading S3; Eq.34)
        const long long pc = ((long long)(g.z + P.pz) * P.ppy + (g.y + 1)) * P.ppx + (g.x + 1);
        const real phi_old = __ldg(Fd.phi_old + pc);
        dtphi = (phi - phi_old) / P.dt;                                        // reading S4
        const real mdot_old = P.rho_g * Fd.pdot[n];
        const real D_old = ux * gx + uy * gy + uz * gz + phi * mdot_old * P.drho;   // reading S5
        pull<LS, real, BC>(Fd.s_in, N, g, P.bc_s, P.bc_T, s);
        T = s[0];
#pragma unroll
        for (int i = 1; i < LS::Q; ++i) T += s[i];
        if (P.latent_heat) T -= P.hdt * P.LCp * (dtphi + D_old);
        // pressure (Eq.28b)
        p = m0 + P.hdt * (P.cs2f * (ux * grx + uy * gry + uz * grz) + rho * P.cs2f * mdot_old * P.drho);
    }

    // ---- H6: production refresh (Eq.18)
    real pdot = real(0);
    if (P.phase_change) {
        const real theta = P.CpL * (T - P.T_sat);
        pdot = P.pc_coef * alpha * (theta - P.theta_I) * phi * (real(1) - phi);
    }
    Fd.pdot[n] = pdot;
    if constexpr (MODE == MODE_STEP_MACRO) {
        Fd.u[n] = ux; Fd.u[N + n] = uy; Fd.u[2 * N + n] = uz;
        Fd.p[n] = p; Fd.T[n] = T;
    }

    // ---- H7: sources, equilibria, BGK (Eq.25): out = (1-om) bar + om eq + dt (1 - om/2) S
    const real mdot = P.rho_g * pdot;
    const real ug = ux * gx + uy * gy + uz * gz;
    const real D = ug + phi * mdot * P.drho;
    const real uu = ux * ux + uy * uy + uz * uz;

    // relaxation rates: tau_bar = nu/(cs2 dt) with harmonic nu (Eq.1b); alpha/(cs2 dt)
    const real den = phi * P.nu_l + (real(1) - phi) * P.nu_g;
    const real om_f = den / (P.nu_prod / (P.cs2f * P.dt) + real(0.5) * den);
    const real om_s = real(1) / (alpha / (P.cs2s * P.dt) + real(0.5));
    const real om_g = P.om_g;

    auto relax = [&](real bar, real eq, real S, real om) -> real {
        if constexpr (MODE == MODE_INIT) return eq + P.hdt * S;   // bar = eq - dt/2 S (Eq.24), reading S9
        else return (real(1) - om) * bar + om * eq + P.dt * (real(1) - real(0.5) * om) * S;
    };

    // -- Navier-Stokes (Eq.26b, 27a-d PAPER.md:198-220)
    {
        const real ic = P.c / P.cs2f;
        const real tx = ux * ic, ty = uy * ic, tz = uz * ic;          // c u / cs2
        const real uu_cs = uu / P.cs2f;
        const real Ax = P.cs2f * grx, Ay = P.cs2f * gry, Az = P.cs2f * grz;   // cs2 grad rho
        const real uA = ux * Ax + uy * Ay + uz * Az;
        const real uF = ux * Fx + uy * Fy + uz * Fz;
        const real cAx = P.c * Ax, cAy = P.c * Ay, cAz = P.c * Az;
        const real cFx = P.c * Fx, cFy = P.c * Fy, cFz = P.c * Fz;
        const real rcs = rho * P.cs2f;
        const real Pf = rcs * mdot * P.drho;                           // Eq.(27c) without w_i
        {   // rest direction
            constexpr real w = real(LF::w(0));
            const real As = -real(0.5) * w * uu_cs;
            const real S = As * (-uA) + (w + As) * (-uF) + w * Pf;
            const real eq = w * p + rcs * As;
            Fd.f_out[n] = relax(MODE == MODE_INIT ? real(0) : f[0], eq, S, om_f);
        }
        static_for<LF::Q>([&](auto icn) {
            constexpr int I = decltype(icn)::value;
            if constexpr (I > 0 && I < LF::opp(I)) {
                constexpr int J = LF::opp(I);
                constexpr real w = real(LF::w(I));
                const real t = dot_e<LF, I, real>(tx, ty, tz);
                const real As = real(0.5) * w * (t * t - uu_cs);
                const real Aa = w * t;
                const real cA = dot_e<LF, I, real>(cAx, cAy, cAz);
                const real cF = dot_e<LF, I, real>(cFx, cFy, cFz);
                const real Gi = As + Aa, Gj = As - Aa;                 // Gamma - w
                const real Si = Gi * (cA - uA) + (w + Gi) * (cF - uF) + w * Pf;
                const real Sj = Gj * (-cA - uA) + (w + Gj) * (-cF - uF) + w * Pf;
                const real eqi = w * p + rcs * Gi, eqj = w * p + rcs * Gj;
                Fd.f_out[(size_t)I * N + n] = relax(MODE == MODE_INIT ? real(0) : f[I], eqi, Si, om_f);
                Fd.f_out[(size_t)J * N + n] = relax(MODE == MODE_INIT ? real(0) : f[J], eqj, Sj, om_f);
            }
        });
    }
    // -- temperature (Eq.33a-d, sign of reading G2)
    {
        const real ic = P.c / P.cs2s;
        const real tx = ux * ic, ty = uy * ic, tz = uz * ic;
        const real uu_cs = uu / P.cs2s;
        const real Qs = P.latent_heat ? -P.LCp * (dtphi + D) : real(0);
        {
            constexpr real w = real(LS::w(0));
            const real G0 = w - real(0.5) * w * uu_cs;
            Fd.s_out[n] = relax(MODE == MODE_INIT ? real(0) : s[0], T * G0, w * Qs, om_s);
        }
        static_for<LS::Q>([&](auto icn) {
            constexpr int I = decltype(icn)::value;
            if constexpr (I > 0 && I < LS::opp(I)) {
                constexpr int J = LS::opp(I);
                constexpr real w = real(LS::w(I));
                const real t = dot_e<LS, I, real>(tx, ty, tz);
                const real Gs = w + real(0.5) * w * (t * t - uu_cs);
                const real Aa = w * t;
                Fd.s_out[(size_t)I * N + n] = relax(MODE == MODE_INIT ? real(0) : s[I], T * (Gs + Aa), w * Qs, om_s);
                Fd.s_out[(size_t)J * N + n] = relax(MODE == MODE_INIT ? real(0) : s[J], T * (Gs - Aa), w * Qs, om_s);
            }
        });
    }
    // -- conservative Allen-Cahn, modified-equilibrium form (Eq.31a,b PAPER.md:246-251; P_i^g Eq.30b)
    {
        real gi[LG::Q];
        if constexpr (MODE != MODE_INIT) pull<LG, real, BC>(Fd.g_in, N, g, P.bc_g, P.bc_phi, gi);
        else {
#pragma unroll
            for (int i = 0; i < LG::Q; ++i) gi[i] = real(0);
        }
        const real ic = P.c / P.cs2g;
        const real tx = ux * ic, ty = uy * ic, tz = uz * ic;
        const real uu_cs = uu / P.cs2g;
        const real inv_norm = rsqrt_(gx * gx + gy * gy + gz * gz + P.eps_n2);     // Eq.(6), reading S7
        const real B = P.cac * phi * (real(1) - phi) * inv_norm;                  // M (4/W) phi(1-phi) c / cs2 / |grad phi|
        const real bx = B * gx, by = B * gy, bz = B * gz;
        {
            constexpr real w = real(LG::w(0));
            const real G0 = w - real(0.5) * w * uu_cs;
            Fd.g_out[n] = relax(MODE == MODE_INIT ? real(0) : gi[0], phi * G0, w * pdot, om_g);
        }
        static_for<LG::Q>([&](auto icn) {
            constexpr int I = decltype(icn)::value;
            if constexpr (I > 0 && I < LG::opp(I)) {
                constexpr int J = LG::opp(I);
                constexpr real w = real(LG::w(I));
                const real t = dot_e<LG, I, real>(tx, ty, tz);
                const real Gs = w + real(0.5) * w * (t * t - uu_cs);
                const real Aa = w * t;
                const real cn = w * dot_e<LG, I, real>(bx, by, bz);
                Fd.g_out[(size_t)I * N + n] = relax(MODE == MODE_INIT ? real(0) : gi[I], phi * (Gs + Aa) + cn, w * pdot, om_g);
                Fd.g_out[(size_t)J * N + n] = relax(MODE == MODE_INIT ? real(0) : gi[J], phi * (Gs - Aa) - cn, w * pdot, om_g);
            }
        });
    }
}

// Direct variant: phi neighbourhood read from global memory through L1.
template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int BZ, int MINB>
__global__ void __launch_bounds__(BX *BY *BZ, MINB)
k_main_direct(const DevParams<real> P, const DevFields<real> Fd) {
    const int t = threadIdx.x;
    const int x0 = blockIdx.x * BX, y0 = blockIdx.y * BY, z0 = blockIdx.z * BZ;
    const int x = x0 + t % BX, y = y0 + (t / BX) % BY, z = z0 + t / (BX * BY);
    if (x >= P.nx || y >= P.ny || z >= P.nz) return;
    const NodeGeom g = make_geom(P, x, y, z);
    PhiGlobal<real> ph{Fd.phi_new + ((long long)(z + P.pz) * P.ppy + (y + 1)) * P.ppx + (x + 1), (long long)P.ppx, P.pplane};
    if (tile_touches_bc(P, x0, y0, z0, BX, BY, BZ)) node_update<LF, LG, LS, real, MODE, true>(P, Fd, g, ph);
    else node_update<LF, LG, LS, real, MODE, false>(P, Fd, g, ph);
}

}  // namespace lbm
