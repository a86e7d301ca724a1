// K_main (steps H2..H7): one thread per lattice node.  Citations are PAPER.md:<line>; readings (G*/S*) are listed in
// DESIGN.md.  Populations are NOT held in registers across the step: the moments are accumulated while the pulled
// values stream in, and every population is read again at the point where it is collided -- from the thread's
// shared-memory column in the default kernel (k_main_smem.cuh), through L1/L2 in the register-gather kernels.  That keeps
// the live state at ~50 doubles: 128 registers, four 128-thread CTAs per SM.
#pragma once

#include "kernels.cuh"
#include "pairs.cuh"

namespace lbm {

// population stores: written once, read by the NEXT step only
template <class sreal, class real> __device__ __forceinline__ void st_pop(sreal *p, real v) {
    *p = sreal(v);
}
// a pair of x-adjacent nodes (pairs.cuh): one 8-byte store; the first node's index is even
__device__ __forceinline__ void st_pop(float *p, f2 v) { *reinterpret_cast<float2 *>(p) = make_float2(v.x, v.y); }
__device__ __forceinline__ void st_pop(float *p, d2 v) { *reinterpret_cast<float2 *>(p) = make_float2((float)v.x, (float)v.y); }

__device__ __forceinline__ double rsqrt_(double a) { return rsqrt(a); }
__device__ __forceinline__ float rsqrt_(float a) { return rsqrtf(a); }
__device__ __forceinline__ f2 rsqrt_(f2 a) { return f2(rsqrtf(a.x), rsqrtf(a.y)); }

// value types of one work item: those of the field arrays, or pairs of them when a thread carries two nodes (real = f2)
template <class real, class Fields> struct NodeTypes { using sreal = typename Fields::sreal; using preal = typename Fields::preal; };
template <class Fields> struct NodeTypes<f2, Fields> { using sreal = float; using preal = d2; };

// a value as the storage type will hold it
template <class sreal, class real> __device__ __forceinline__ real as_stored(real v) { return real(sreal(v)); }
template <class sreal> __device__ __forceinline__ f2 as_stored(f2 v) { return v; }   // float storage of float pairs

// Source of one node's inputs, direct variant: gathers straight from global memory (pull with wrap / boundary
// rules); the phi^{n+1} neighbourhood comes from the padded array through L1/L2.
template <class LF, class LG, class LS, class real, bool BC, class Fields = DevFields<real>> struct SrcGlobal {
    using preal = typename Fields::preal;
    const DevParams<real> &P;
    const Fields &Fd;
    const NodeGeom &g;
    const preal *__restrict__ pc;   // the node's own element of the padded phi^{n+1}
    unsigned pcoff;
    __device__ __forceinline__ SrcGlobal(const DevParams<real> &P_, const Fields &Fd_, const NodeGeom &g_)
        : P(P_), Fd(Fd_), g(g_) {
        pcoff = ((unsigned)(g.z + P.pz) * (unsigned)P.ppy + (unsigned)(g.y + 1)) * (unsigned)P.ppx + (unsigned)(g.x + P.xpad);
        pc = Fd.phi_new + pcoff;
    }
    __device__ __forceinline__ void pops_ready() const {}
    __device__ __forceinline__ void f_ready() const {}
    __device__ __forceinline__ void phi_ready() const {}
    __device__ __forceinline__ preal phi(int dx, int dy, int dz) const { return __ldg(pc + (dx + dy * P.ppx + dz * (int)P.pplane)); }
    __device__ __forceinline__ preal phi_old() const { return __ldg(Fd.phi_old + pcoff); }
    __device__ __forceinline__ real pdot_old() const { return real(Fd.pdot_in[g.n]); }
    // AGAIN = true: second read of a value already read for the moments (see ld_again)
    template <int I, bool AGAIN = false> __device__ __forceinline__ real f() const { return pull_one<LF, I, real, BC, AGAIN>(Fd.f_in, (unsigned)P.N, g, P.bc_f, P.bc_p); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real s() const { return pull_one<LS, I, real, BC, AGAIN>(Fd.s_in, (unsigned)P.N, g, P.bc_s, P.bc_T); }
    template <int I, bool AGAIN = false> __device__ __forceinline__ real gg() const { return pull_one<LG, I, real, BC, AGAIN>(Fd.g_in, (unsigned)P.N, g, P.bc_g, P.bc_phi); }
    // ---- variant modes only ----
    // phi^{n+1} up to two nodes away (second neighbour of the second-order biased difference), with the ghost
    // rule of reading S8-iv carried two layers deep: periodic image; zero-flux mirror; Dirichlet 2 v - mirror
    __device__ __forceinline__ preal phi_far(int dx, int dy, int dz) const {
        int q[3] = {g.x + dx, g.y + dy, g.z + dz}, cross[3];
        ghost_source(P, P.bc_g, q, cross);
        preal v = __ldg(Fd.phi_new + ((unsigned)(q[2] + P.pz) * (unsigned)P.ppy + (unsigned)(q[1] + 1)) * (unsigned)P.ppx + (unsigned)(q[0] + P.xpad));
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (cross[a] && P.bc_g[a][cross[a] - 1] == BC_ANTI) v = preal(2) * preal(P.bc_phi[a][cross[a] - 1]) - v;
        return v;
    }
    // component `comp` of the velocity array at a neighbour (stencil divergence, reading S17): periodic image; odd
    // reflection in a no-slip wall (zero on the wall); even reflection in an open face
    __device__ __forceinline__ real u_nb(int comp, int dx, int dy, int dz) const {
        int q[3] = {g.x + dx, g.y + dy, g.z + dz}, cross[3];
        ghost_source(P, P.bc_f, q, cross);
        real v = real(Fd.u[(unsigned)comp * (unsigned)P.N + ((unsigned)q[2] * (unsigned)P.ny + (unsigned)q[1]) * (unsigned)P.nx + (unsigned)q[0]]);
#pragma unroll
        for (int a = 0; a < 3; ++a)
            if (cross[a] && P.bc_f[a][cross[a] - 1] == BC_BOUNCE) v = -v;
        return v;
    }
};

// Geom: NodeGeom, or NodeGeom2 for a pair of nodes (k_main_pair.cuh) -- only the linear index n of the (first) node is used here.
template <class LF, class LG, class LS, class real, int MODE, class Src, class Fields, class Geom>
__device__ __forceinline__ void node_update(const DevParams<real> &P, const Fields &Fd, const Geom &g,
                                            const Src &src) {
    using sreal = typename NodeTypes<real, Fields>::sreal;
    using preal = typename NodeTypes<real, Fields>::preal;   // phi arrays; differences of phi are taken in this type, then narrowed
    const unsigned n = g.n;
    const unsigned N = (unsigned)P.N;

    // ---- H5 (first half): zeroth moment of s.  Loaded first so that these loads are in flight during the stencil.
    src.pops_ready();   // staged variants: the node's asynchronous copies have landed
    real sum_s = real(0);
    if constexpr (!mode_is_init<MODE>::value) {
        static_for<LS::Q>([&](auto ic) { sum_s += src.template s<decltype(ic)::value>(); });
    }

    // ---- H2: grad phi, lap phi by directional derivatives on the NS lattice (Eq.35a,b 36a,b; PAPER.md:291-315;
    //      the printed factor 3 is 1/e2, reading S2).  Opposite directions are paired: one difference, one sum.
    src.phi_ready();   // TMA-staged phi tile: wait here, after the s loads have been issued
    const preal phi_p = src.phi(0, 0, 0);
    const real phi = real(phi_p);
    real gx = real(0), gy = real(0), gz = real(0), lsum = real(0);
    static_for<LF::Q>([&](auto ic) {
        constexpr int I = decltype(ic)::value;
        if constexpr (I > 0 && I < LF::opp(I)) {
            constexpr int ex = LF::ex(I), ey = LF::ey(I), ez = LF::ez(I);
            const preal pp = src.phi(ex, ey, ez), pm = src.phi(-ex, -ey, -ez);
            real d = real(pp - pm);   // central difference Eq.(35a), the pair (e, -e) at once
            if constexpr (mode_has_variants<MODE>::value) {
                // biased differences of PAPER.md:318 inside Eq.(35b), again both directions of the pair
                if (P.grad_scheme == 1) d = real((pp - phi_p) - (pm - phi_p));
                else if (P.grad_scheme == 2) {
                    const preal pp2 = src.phi_far(2 * ex, 2 * ey, 2 * ez), pm2 = src.phi_far(-2 * ex, -2 * ey, -2 * ez);
                    d = real(preal(0.5) * ((preal(4) * pp - pp2 - preal(3) * phi_p) - (preal(4) * pm - pm2 - preal(3) * phi_p)));
                }
            }
            constexpr real w = real(LF::w(I));
            if constexpr (ex != 0) gx += (ex > 0 ? w : -w) * d;
            if constexpr (ey != 0) gy += (ey > 0 ? w : -w) * d;
            if constexpr (ez != 0) gz += (ez > 0 ? w : -w) * d;
            lsum += w * real(pp + pm);
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
    const real Fx = mu * gx + bu * P.grav[0] + P.force[0];                     // Eq.(12),(13) PAPER.md:106-114; body force PAPER.md:418
    const real Fy = mu * gy + bu * P.grav[1] + P.force[1];
    const real Fz = mu * gz + bu * P.grav[2] + P.force[2];
    const real grx = P.rho_diff * gx, gry = P.rho_diff * gy, grz = P.rho_diff * gz;   // grad rho
    const real alpha = P.alpha_l + phi * P.alpha_diff;                         // reading S6
    // relaxation rates: tau_bar = nu/(cs2 dt) with harmonic nu (Eq.1b); alpha/(cs2 dt);
    // om = 1/(tau_bar + 1/2) (Eq.25).  om_f = den/(nu_l nu_g/(cs2 dt) + den/2), den = phi nu_l + (1-phi) nu_g.
    // The three per-node divisions (1/rho, om_f, om_s) share ONE reciprocal: 1/(rho * df * ds).
    const real den = phi * P.nu_l + (real(1) - phi) * P.nu_g;
    const real df = P.tauf_num + real(0.5) * den;
    const real ds = alpha * P.taus_den + real(0.5);
    const real rds = rho * ds;
    const real rall = real(1) / (rds * df);
    const real inv_rho = rall * ds * df;
    const real om_f = den * (rall * rds);
    const real om_s = rall * (rho * df);

    // variant modes, div_scheme = stencil: div(u phi) by Eq.(35a,b) on the components of u phi, from the velocity ARRAY
    // (this level's u of every node: the input at initialisation, written by the MODE_U pass before a step) -- reading S17
    real D_st = real(0);
    bool use_st = false;
    if constexpr (MODE == MODE_INIT_VAR || MODE == MODE_STEP_VAR) {
        if (P.div_scheme) {
            use_st = true;
            static_for<LF::Q>([&](auto ic) {
                constexpr int I = decltype(ic)::value;
                if constexpr (I > 0 && I < LF::opp(I)) {
                    constexpr int ex = LF::ex(I), ey = LF::ey(I), ez = LF::ez(I);
                    real up = real(0), um = real(0);
                    if constexpr (ex != 0) { up += real(ex) * src.u_nb(0, ex, ey, ez); um += real(ex) * src.u_nb(0, -ex, -ey, -ez); }
                    if constexpr (ey != 0) { up += real(ey) * src.u_nb(1, ex, ey, ez); um += real(ey) * src.u_nb(1, -ex, -ey, -ez); }
                    if constexpr (ez != 0) { up += real(ez) * src.u_nb(2, ex, ey, ez); um += real(ez) * src.u_nb(2, -ex, -ey, -ez); }
                    D_st += real(LF::w(I)) * (up * real(src.phi(ex, ey, ez)) - um * real(src.phi(-ex, -ey, -ez)));
                }
            });
            D_st *= P.inv_dx * real(1.0 / LF::e2);
        }
    }

    real ux, uy, uz, p, T, dtphi;
    real pd_old = real(0);   // production rate of the previous level: in the moment corrections and folded into the stored g_0
    if constexpr (mode_is_init<MODE>::value) {
        ux = real(Fd.u[n]); uy = real(Fd.u[N + n]); uz = (LF::D == 3) ? real(Fd.u[2 * N + n]) : real(0);
        p = real(Fd.p[n]); T = real(Fd.T[n]); dtphi = real(0);
    } else {
        // ---- H4: NS moments (Eq.28a), accumulated as the pulled values arrive
        real m0 = real(0), mx = real(0), my = real(0), mz = real(0);
        src.f_ready();   // staged variants: the second group of copies (f, g) has landed
        static_for<LF::Q>([&](auto ic) {
            constexpr int I = decltype(ic)::value;
            const real fi = src.template f<I>();
            m0 += fi;
            if constexpr (LF::ex(I) != 0) mx += LF::ex(I) > 0 ? fi : -fi;
            if constexpr (LF::ey(I) != 0) my += LF::ey(I) > 0 ? fi : -fi;
            if constexpr (LF::ez(I) != 0) mz += LF::ez(I) > 0 ? fi : -fi;
        });
        const real cm = P.c_cs2f;
        ux = (cm * mx + P.hdt * Fx) * inv_rho;
        uy = (cm * my + P.hdt * Fy) * inv_rho;
        uz = (cm * mz + P.hdt * Fz) * inv_rho;
        if constexpr (MODE == MODE_STEP_PU) {   // Zalesak / vortex verifications: u is the field given at init
            ux = real(Fd.u[n]); uy = real(Fd.u[N + n]); uz = (LF::D == 3) ? real(Fd.u[2 * N + n]) : real(0);
        }
        if constexpr (MODE == MODE_U) {         // velocity pass: u^{n+1} of this node for its neighbours' stencil divergence
            st_pop(Fd.u + n, ux); st_pop(Fd.u + (N + n), uy);
            if constexpr (LF::D == 3) st_pop(Fd.u + (2 * N + n), uz);
            return;
        }
        if constexpr (MODE == MODE_STEP_VAR) {  // prescribed, or already in the array (the value the neighbours saw)
            if (P.prescribed_u || P.div_scheme) {
                ux = real(Fd.u[n]); uy = real(Fd.u[N + n]); uz = (LF::D == 3) ? real(Fd.u[2 * N + n]) : real(0);
            }
        }
        // ---- H1 (time derivative), H5: heat moment with the STORED production rate (reading S3; Eq.34)
        dtphi = real(phi_p - src.phi_old()) * P.inv_dt;                              // reading S4
        pd_old = src.pdot_old();
        const real mdot_old = P.rho_g * pd_old;
        const real D_old = use_st ? D_st : ux * gx + uy * gy + uz * gz + phi * mdot_old * P.drho;   // reading S5 (or S17)
        T = sum_s;
        if (P.latent_heat) T -= P.hdt * P.LCp * (dtphi + D_old);
        // pressure (Eq.28b)
        p = m0 + P.hdt * (P.cs2f * (ux * grx + uy * gry + uz * grz) + rho * P.cs2f * mdot_old * P.drho);
    }

    // ---- H6: production refresh (Eq.18)
    real pdot = real(0);
    if (P.phase_change) {
        const real theta = P.CpL * (T - P.T_sat);
        // this level's collision and the next level's moment corrections use the SAME value (reading S3): the stored one
        pdot = as_stored<sreal>(real(P.pc_coef * alpha * (theta - P.theta_I) * phi * (real(1) - phi)));
    }
    st_pop(Fd.pdot + n, pdot);
    if constexpr (MODE == MODE_STEP_MACRO) {
        st_pop(Fd.u + n, ux); st_pop(Fd.u + (N + n), uy); st_pop(Fd.u + (2 * N + n), uz);
        st_pop(Fd.p + n, p); st_pop(Fd.T + n, T);
    }
    if constexpr (MODE == MODE_STEP_PU) { st_pop(Fd.p + n, p); st_pop(Fd.T + n, T); }
    if constexpr (MODE == MODE_STEP_VAR) {
        st_pop(Fd.p + n, p); st_pop(Fd.T + n, T);
        if (!(P.prescribed_u || P.div_scheme)) { st_pop(Fd.u + n, ux); st_pop(Fd.u + (N + n), uy); st_pop(Fd.u + (2 * N + n), uz); }
    }

    // ---- H7: sources, equilibria, BGK (Eq.25)
    const real mdot = P.rho_g * pdot;
    const real ug = ux * gx + uy * gy + uz * gz;
    const real D = use_st ? D_st : ug + phi * mdot * P.drho;
    const real uu = ux * ux + uy * uy + uz * uz;

    // BGK with the source shift folded in: out_i = a bar_i + om eq_i + b S_i, with (a, om, b) = (1-om, om, dt(1-om/2)),
    // or (0, 1, dt/2) at initialisation where bar = eq - dt/2 S (Eq.24, reading S9).
    //
    // -- Navier-Stokes (Eq.26b, 27a-d PAPER.md:198-220).  With Gamma_i - w_i = w_i (q +- t), t = c_i.u/cs2,
    //    q = t^2/2 - u.u/(2 cs2), A = cs2 grad rho, H = A + F_tot, mdot = mass production rate:
    //      eq_i = w_i p + rho cs2 (Gamma_i - w_i)
    //      S_i  = (Gamma_i - w_i)(c_i.H - u.H) + w_i (c_i.F - u.F + rho cs2 mdot Drho)
    //    so out_i = a bar_i + (Gamma_i - w_i)(K1 + b c_i.H) + w_i (K2 + b c_i.F),
    //    K1 = om rho cs2 - b u.H,  K2 = om p + b (rho cs2 mdot Drho - u.F).
    {
        const real om = mode_is_init<MODE>::value ? real(1) : om_f;
        const real a = mode_is_init<MODE>::value ? real(0) : real(1) - om_f;
        const real b = mode_is_init<MODE>::value ? P.hdt : P.dt * (real(1) - real(0.5) * om_f);
        const real ic = P.c_cs2f;
        const real tx = ux * ic, ty = uy * ic, tz = uz * ic;          // c u / cs2
        const real U = real(-0.5) * uu * P.inv_cs2f;
        const real rcs = rho * P.cs2f;
        const real Hx = P.cs2f * grx + Fx, Hy = P.cs2f * gry + Fy, Hz = P.cs2f * grz + Fz;
        const real K1 = om * rcs - b * (ux * Hx + uy * Hy + uz * Hz);
        const real K2 = om * p + b * (rcs * mdot * P.drho - (ux * Fx + uy * Fy + uz * Fz));
        const real bc = b * P.c;
        const real Hbx = bc * Hx, Hby = bc * Hy, Hbz = bc * Hz;
        const real Fbx = bc * Fx, Fby = bc * Fy, Fbz = bc * Fz;
        {   // rest direction: t = 0
            constexpr real w = real(LF::w(0));
            real bar = real(0);
            if constexpr (!mode_is_init<MODE>::value) bar = src.template f<0, true>();
            st_pop(Fd.f_out + (n), a * bar + w * (U * K1 + K2));
        }
        static_for<LF::Q>([&](auto icn) {
            constexpr int I = decltype(icn)::value;
            if constexpr (I > 0 && I < LF::opp(I)) {
                constexpr int J = LF::opp(I);
                constexpr real w = real(LF::w(I));
                real bi = real(0), bj = real(0);
                if constexpr (!mode_is_init<MODE>::value) { bi = src.template f<I, true>(); bj = src.template f<J, true>(); }
                const real t = dot_e<LF, I, real>(tx, ty, tz);
                const real q = real(0.5) * t * t + U;
                const real h = dot_e<LF, I, real>(Hbx, Hby, Hbz);
                const real fb = dot_e<LF, I, real>(Fbx, Fby, Fbz);
                st_pop(Fd.f_out + ((unsigned)I * N + n), a * bi + w * ((q + t) * (K1 + h) + (K2 + fb)));
                st_pop(Fd.f_out + ((unsigned)J * N + n), a * bj + w * ((q - t) * (K1 - h) + (K2 - fb)));
            }
        });
    }
    // -- temperature (Eq.33a-d, sign of reading G2): eq_i = T Gamma_i, S_i = -w_i (L/Cp)(dphi/dt + D)
    {
        const real om = mode_is_init<MODE>::value ? real(1) : om_s;
        const real a = mode_is_init<MODE>::value ? real(0) : real(1) - om_s;
        const real b = mode_is_init<MODE>::value ? P.hdt : P.dt * (real(1) - real(0.5) * om_s);
        const real ic = P.c_cs2s;
        const real tx = ux * ic, ty = uy * ic, tz = uz * ic;
        const real U1 = real(1) - real(0.5) * uu * P.inv_cs2s;
        const real TO = om * T;
        const real bQ = P.latent_heat ? -b * P.LCp * (dtphi + D) : real(0);
        {
            constexpr real w = real(LS::w(0));
            real bar = real(0);
            if constexpr (!mode_is_init<MODE>::value) bar = src.template s<0, true>();
            st_pop(Fd.s_out + (n), a * bar + w * (TO * U1 + bQ));
        }
        static_for<LS::Q>([&](auto icn) {
            constexpr int I = decltype(icn)::value;
            if constexpr (I > 0 && I < LS::opp(I)) {
                constexpr int J = LS::opp(I);
                constexpr real w = real(LS::w(I));
                real bi = real(0), bj = real(0);
                if constexpr (!mode_is_init<MODE>::value) { bi = src.template s<I, true>(); bj = src.template s<J, true>(); }
                const real t = dot_e<LS, I, real>(tx, ty, tz);
                const real q = real(0.5) * t * t + U1;
                st_pop(Fd.s_out + ((unsigned)I * N + n), a * bi + w * (TO * (q + t) + bQ));
                st_pop(Fd.s_out + ((unsigned)J * N + n), a * bj + w * (TO * (q - t) + bQ));
            }
        });
    }
    // -- conservative Allen-Cahn, modified-equilibrium form (Eq.31a,b PAPER.md:246-251; P_i^g Eq.30b):
    //    eq_i = phi Gamma_i + M (4/W) phi (1-phi) w_i c_i.n / cs2,  S_i = w_i Pdot
    //    Evaluated in the type of the phi arrays (greal = preal): sum_i g*_i is the phi of the next level, and what its
    //    rounding adds to dphi/dt reaches T multiplied by L/Cp.
    {
        using greal = preal;
        const greal om_g = greal(P.g_om), dtg = greal(P.g_dt);   // constants carried in double: no widening per node
        const greal om = mode_is_init<MODE>::value ? greal(1) : om_g;
        const greal a = mode_is_init<MODE>::value ? greal(0) : greal(1) - om_g;
        const greal b = mode_is_init<MODE>::value ? greal(0.5) * dtg : dtg * (greal(1) - greal(0.5) * om_g);
        const greal ic = greal(P.g_c_cs2);
        const greal tx = greal(ux) * ic, ty = greal(uy) * ic, tz = greal(uz) * ic;
        const greal U1 = greal(1) - greal(0.5) * greal(uu) * greal(P.g_inv_cs2);
        const real inv_norm = rsqrt_(gx * gx + gy * gy + gz * gz + P.eps_n2);     // Eq.(6), reading S7
        const greal phi_g = greal(phi_p);
        const greal B = om * greal(P.g_cac) * phi_g * (greal(1) - phi_g) * greal(inv_norm);   // om M (4/W) phi(1-phi) c / cs2 / |grad phi|
        const greal bx = B * greal(gx), by = B * greal(gy), bz = B * greal(gz);
        const greal PO = om * phi_g;
        const greal bP = b * greal(pdot);
        {
            // The rest population never moves, so the term dt/2 Pdot of Eq.(32) (phi^{n+1} = sum_i g_i + dt/2 Pdot, same node,
            // same production rate as stored below) rides in it: stored g_0' = g*_0 + dt/2 Pdot.  K_phi then needs no Pdot, and
            // the bar value is recovered here with the production rate of the previous level.
            constexpr greal w = greal(LG::w(0));
            const greal hdtg = greal(0.5) * dtg;
            greal bar = greal(0);
            if constexpr (!mode_is_init<MODE>::value) bar = greal(src.template gg<0>()) - hdtg * greal(pd_old);
            st_pop(Fd.g_out + (n), a * bar + w * (PO * U1 + bP) + hdtg * greal(pdot));
        }
        static_for<LG::Q>([&](auto icn) {
            constexpr int I = decltype(icn)::value;
            if constexpr (I > 0 && I < LG::opp(I)) {
                constexpr int J = LG::opp(I);
                constexpr greal w = greal(LG::w(I));
                greal bi = greal(0), bj = greal(0);
                if constexpr (!mode_is_init<MODE>::value) { bi = greal(src.template gg<I>()); bj = greal(src.template gg<J>()); }
                const greal t = dot_e<LG, I, greal>(tx, ty, tz);
                const greal q = greal(0.5) * t * t + U1;
                const greal cn = dot_e<LG, I, greal>(bx, by, bz);
                st_pop(Fd.g_out + ((unsigned)I * N + n), a * bi + w * (PO * (q + t) + (bP + cn)));
                st_pop(Fd.g_out + ((unsigned)J * N + n), a * bj + w * (PO * (q - t) + (bP - cn)));
            }
        });
    }
}

// Direct variant: everything gathered from global memory.
template <class LF, class LG, class LS, class real, int MODE, int BX, int BY, int BZ, int MINB, class Fields>
__global__ void __launch_bounds__(BX *BY *BZ, MINB)
k_main_direct(const DevParams<real> P, const Fields Fd) {
    const int t = threadIdx.x;
    const int x0 = blockIdx.x * BX;
    int y0, z0;
    tile_origin<LF::D>(P, BY, BZ, y0, z0);
    const int x = x0 + t % BX, y = y0 + (t / BX) % BY, z = z0 + t / (BX * BY);
    if (!node_active<LF::D>(P, x, y, z)) return;
    const NodeGeom g = make_geom(P, x, y, z);
    if (tile_touches_bc(P, x0, y0, z0, BX, BY, BZ)) {
        const SrcGlobal<LF, LG, LS, real, true, Fields> src(P, Fd, g);
        node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
    } else {
        const SrcGlobal<LF, LG, LS, real, false, Fields> src(P, Fd, g);
        node_update<LF, LG, LS, real, MODE>(P, Fd, g, src);
    }
}

}  // namespace lbm
