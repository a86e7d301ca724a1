/*
 * CPU ORACLE -- TEST INFRASTRUCTURE ONLY (see lbm_oracle.h for the rules).
 *
 * One time step n -> n+1 is five separate passes over the lattice, in the paper's order:
 *   P1 derive   : grad phi (Eq.35a,b), lap phi (Eq.36a,b)
 *   P2+P3 collide: closures (1a,1b,6,12,13,14,18), Gamma_i (27d), equilibria and sources of the three
 *                 lattices (26b,27a-c ; 31b,30b or 29b,30a-b ; 33b-d), BGK Eq.(25)
 *   P4 stream   : pull streaming with periodic wrap, half bounce-back,
 *                 anti-bounce-back
 *   P5 moments  : Eq.(32), (28a), (34), (28b), then refresh of Eq.(18)
 * State kept between steps: streamed populations, phi, u, p, T, dphi/dt and the production field Pdot.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no fast-math, no FMA contraction).
 */
#include "lbm_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QMAX 19

typedef struct {
    int Q;
    int e[QMAX][3];
    double w[QMAX];
    int opp[QMAX];
    double e2; /* lattice constant: c_s^2 = e2 * c^2 */
} lattice_t;

struct oracle_ctx {
    oracle_params P;
    long N;
    lattice_t Lf, Lg, Ls;
    int cac_form;
    long nsteps;
    /* host constants, Eq.(15b): K = 3/2 W sigma, H = 12 sigma / W */
    double K, H;
    /* streamed populations (level n) and post-collision populations */
    double *f, *g, *s, *fpost, *gpost, *spost;
    /* macroscopic fields at level n */
    double *phi, *phi_prev, *dtphi, *u, *p, *T, *pdot;
    /* prescribed-velocity mode: u of the NEXT time level, given by oracle_set_velocity (NULL: u does not change) */
    double *u_next;
    /* derived fields of phi at level n */
    double *grad, *lap;
    /* ORA_DIV_STENCIL: div(u phi) at level n by the directional-derivative stencil (else NULL) */
    double *divuphi;
};

/* ------------------------------------------------------------------------------------------------
 * Lattices.  PAPER.md:190.  D2Q9 weights are the standard ones (not printed in the paper, S1);
 * D2Q5 is not in the paper (S1): w0 = 1/3, w1..4 = 1/6, e2 = 1/3.
 * D3Q7 / D3Q19 vector order: the paper abbreviates the lists with "..." (G7); the order used is
 * e1=(1,0,0) e2=(0,1,0) e3=(0,0,1) e4=(-1,0,0) e5=(0,-1,0) e6=(0,0,-1), then the pairs the paper
 * prints: e7,8=(+-1,1,0) e9,10=(+-1,-1,0) e11,12=(+-1,0,1) e13,14=(+-1,0,-1) e15,16=(0,+-1,1)
 * e17,18=(0,+-1,-1).
 * ---------------------------------------------------------------------------------------------- */
static void set_e(lattice_t *L, int i, int ex, int ey, int ez, double w)
{
    L->e[i][0] = ex; L->e[i][1] = ey; L->e[i][2] = ez; L->w[i] = w;
}

static int make_lattice(int id, lattice_t *L)
{
    memset(L, 0, sizeof(*L));
    switch (id) {
    case ORA_D2Q5:
        L->Q = 5; L->e2 = 1.0 / 3.0;
        set_e(L, 0, 0, 0, 0, 1.0 / 3.0);
        set_e(L, 1, 1, 0, 0, 1.0 / 6.0); set_e(L, 2, 0, 1, 0, 1.0 / 6.0);
        set_e(L, 3, -1, 0, 0, 1.0 / 6.0); set_e(L, 4, 0, -1, 0, 1.0 / 6.0);
        break;
    case ORA_D2Q9:
        L->Q = 9; L->e2 = 1.0 / 3.0;
        set_e(L, 0, 0, 0, 0, 4.0 / 9.0);
        set_e(L, 1, 1, 0, 0, 1.0 / 9.0); set_e(L, 2, 0, 1, 0, 1.0 / 9.0);
        set_e(L, 3, -1, 0, 0, 1.0 / 9.0); set_e(L, 4, 0, -1, 0, 1.0 / 9.0);
        set_e(L, 5, 1, 1, 0, 1.0 / 36.0); set_e(L, 6, -1, 1, 0, 1.0 / 36.0);
        set_e(L, 7, -1, -1, 0, 1.0 / 36.0); set_e(L, 8, 1, -1, 0, 1.0 / 36.0);
        break;
    case ORA_D3Q7:
        L->Q = 7; L->e2 = 1.0 / 4.0;
        set_e(L, 0, 0, 0, 0, 1.0 / 4.0);
        set_e(L, 1, 1, 0, 0, 1.0 / 8.0); set_e(L, 2, 0, 1, 0, 1.0 / 8.0); set_e(L, 3, 0, 0, 1, 1.0 / 8.0);
        set_e(L, 4, -1, 0, 0, 1.0 / 8.0); set_e(L, 5, 0, -1, 0, 1.0 / 8.0); set_e(L, 6, 0, 0, -1, 1.0 / 8.0);
        break;
    case ORA_D3Q19:
        L->Q = 19; L->e2 = 1.0 / 3.0;
        set_e(L, 0, 0, 0, 0, 1.0 / 3.0);
        set_e(L, 1, 1, 0, 0, 1.0 / 18.0); set_e(L, 2, 0, 1, 0, 1.0 / 18.0); set_e(L, 3, 0, 0, 1, 1.0 / 18.0);
        set_e(L, 4, -1, 0, 0, 1.0 / 18.0); set_e(L, 5, 0, -1, 0, 1.0 / 18.0); set_e(L, 6, 0, 0, -1, 1.0 / 18.0);
        set_e(L, 7, 1, 1, 0, 1.0 / 36.0); set_e(L, 8, -1, 1, 0, 1.0 / 36.0);
        set_e(L, 9, 1, -1, 0, 1.0 / 36.0); set_e(L, 10, -1, -1, 0, 1.0 / 36.0);
        set_e(L, 11, 1, 0, 1, 1.0 / 36.0); set_e(L, 12, -1, 0, 1, 1.0 / 36.0);
        set_e(L, 13, 1, 0, -1, 1.0 / 36.0); set_e(L, 14, -1, 0, -1, 1.0 / 36.0);
        set_e(L, 15, 0, 1, 1, 1.0 / 36.0); set_e(L, 16, 0, -1, 1, 1.0 / 36.0);
        set_e(L, 17, 0, 1, -1, 1.0 / 36.0); set_e(L, 18, 0, -1, -1, 1.0 / 36.0);
        break;
    case ORA_D3Q15:
        /* e7 = (1,1,1), e8 = (-1,1,1), "...", e14 = (1,-1,-1); the elided ones are taken counter-clockwise
         * around z on each level, which ends on the printed e14 (reading G10).  w0 = 2/9, w1..6 = 1/9, w7..14 = 1/72. */
        L->Q = 15; L->e2 = 1.0 / 3.0;
        set_e(L, 0, 0, 0, 0, 2.0 / 9.0);
        set_e(L, 1, 1, 0, 0, 1.0 / 9.0); set_e(L, 2, 0, 1, 0, 1.0 / 9.0); set_e(L, 3, 0, 0, 1, 1.0 / 9.0);
        set_e(L, 4, -1, 0, 0, 1.0 / 9.0); set_e(L, 5, 0, -1, 0, 1.0 / 9.0); set_e(L, 6, 0, 0, -1, 1.0 / 9.0);
        set_e(L, 7, 1, 1, 1, 1.0 / 72.0); set_e(L, 8, -1, 1, 1, 1.0 / 72.0);
        set_e(L, 9, -1, -1, 1, 1.0 / 72.0); set_e(L, 10, 1, -1, 1, 1.0 / 72.0);
        set_e(L, 11, 1, 1, -1, 1.0 / 72.0); set_e(L, 12, -1, 1, -1, 1.0 / 72.0);
        set_e(L, 13, -1, -1, -1, 1.0 / 72.0); set_e(L, 14, 1, -1, -1, 1.0 / 72.0);
        break;
    default:
        return -1;
    }
    for (int i = 0; i < L->Q; ++i) {
        L->opp[i] = -1;
        for (int j = 0; j < L->Q; ++j)
            if (L->e[j][0] == -L->e[i][0] && L->e[j][1] == -L->e[i][1] && L->e[j][2] == -L->e[i][2])
                L->opp[i] = j;
        if (L->opp[i] < 0) return -1;
    }
    return 0;
}

int oracle_lattice(int id, int *e, double *w, double *e2)
{
    lattice_t L;
    if (make_lattice(id, &L)) return -1;
    for (int i = 0; i < L.Q; ++i) {
        if (e) { e[3 * i] = L.e[i][0]; e[3 * i + 1] = L.e[i][1]; e[3 * i + 2] = L.e[i][2]; }
        if (w) w[i] = L.w[i];
    }
    if (e2) *e2 = L.e2;
    return L.Q;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int lattice_is_3d(int id) { return id == ORA_D3Q7 || id == ORA_D3Q19 || id == ORA_D3Q15; }

static long idx(const oracle_ctx *c, int x, int y, int z)
{
    return ((long)z * c->P.ny + y) * c->P.nx + x;
}

static int axis_len(const oracle_ctx *c, int a) { return a == 0 ? c->P.nx : (a == 1 ? c->P.ny : c->P.nz); }

oracle_ctx *oracle_create(const oracle_params *p)
{
    if (!p) return NULL;
    if (p->nx < 1 || p->ny < 1 || p->nz < 1) return NULL;
    if (!(p->dx > 0) || !(p->dt > 0) || !(p->W > 0) || !(p->rho_l > 0) || !(p->rho_g > 0)) return NULL;
    if (!(p->nu_l > 0) || !(p->nu_g > 0) || !(p->M > 0) || !(p->alpha_l > 0) || !(p->alpha_g > 0)) return NULL;
    if (!(p->Cp > 0) || p->L_latent == 0.0 || !(p->A > 0)) return NULL;
    if (p->grad_scheme < ORA_GRAD_CENTRAL || p->grad_scheme > ORA_GRAD_BIASED2) return NULL;
    if (p->div_scheme < ORA_DIV_PRODUCT || p->div_scheme > ORA_DIV_STENCIL) return NULL;
    oracle_ctx *c = (oracle_ctx *)calloc(1, sizeof(*c));
    if (!c) return NULL;
    c->P = *p;
    if (make_lattice(p->lat_f, &c->Lf) || make_lattice(p->lat_g, &c->Lg) || make_lattice(p->lat_s, &c->Ls)) {
        free(c); return NULL;
    }
    int three_d = p->nz > 1;
    if (lattice_is_3d(p->lat_f) != three_d || lattice_is_3d(p->lat_g) != three_d ||
        lattice_is_3d(p->lat_s) != three_d) { free(c); return NULL; }
    for (int a = 0; a < 3; ++a) {
        /* a periodic face must be paired with a periodic face, for every distribution */
        if ((p->bc_f[a][0] == ORA_F_PERIODIC) != (p->bc_f[a][1] == ORA_F_PERIODIC) ||
            (p->bc_g[a][0] == ORA_S_PERIODIC) != (p->bc_g[a][1] == ORA_S_PERIODIC) ||
            (p->bc_s[a][0] == ORA_S_PERIODIC) != (p->bc_s[a][1] == ORA_S_PERIODIC)) { free(c); return NULL; }
        if ((p->bc_f[a][0] == ORA_F_PERIODIC) != (p->bc_g[a][0] == ORA_S_PERIODIC) ||
            (p->bc_f[a][0] == ORA_F_PERIODIC) != (p->bc_s[a][0] == ORA_S_PERIODIC)) { free(c); return NULL; }
    }
    c->N = (long)p->nx * p->ny * p->nz;
    c->K = 1.5 * p->W * p->sigma;  /* Eq.(15b) */
    c->H = 12.0 * p->sigma / p->W; /* Eq.(15b) */
    c->cac_form = ORA_CAC_MODIFIED_EQ;
    long N = c->N;
    c->f = (double *)calloc((size_t)c->Lf.Q * N, sizeof(double));
    c->g = (double *)calloc((size_t)c->Lg.Q * N, sizeof(double));
    c->s = (double *)calloc((size_t)c->Ls.Q * N, sizeof(double));
    c->fpost = (double *)calloc((size_t)c->Lf.Q * N, sizeof(double));
    c->gpost = (double *)calloc((size_t)c->Lg.Q * N, sizeof(double));
    c->spost = (double *)calloc((size_t)c->Ls.Q * N, sizeof(double));
    c->phi = (double *)calloc(N, sizeof(double));
    c->phi_prev = (double *)calloc(N, sizeof(double));
    c->dtphi = (double *)calloc(N, sizeof(double));
    c->u = (double *)calloc(3 * N, sizeof(double));
    c->p = (double *)calloc(N, sizeof(double));
    c->T = (double *)calloc(N, sizeof(double));
    c->pdot = (double *)calloc(N, sizeof(double));
    c->grad = (double *)calloc(3 * N, sizeof(double));
    c->lap = (double *)calloc(N, sizeof(double));
    if (p->div_scheme == ORA_DIV_STENCIL) {
        c->divuphi = (double *)calloc(N, sizeof(double));
        if (!c->divuphi) { oracle_destroy(c); return NULL; }
    }
    if (!c->f || !c->g || !c->s || !c->fpost || !c->gpost || !c->spost || !c->phi || !c->phi_prev ||
        !c->dtphi || !c->u || !c->p || !c->T || !c->pdot || !c->grad || !c->lap) {
        oracle_destroy(c); return NULL;
    }
    return c;
}

void oracle_destroy(oracle_ctx *c)
{
    if (!c) return;
    free(c->f); free(c->g); free(c->s); free(c->fpost); free(c->gpost); free(c->spost);
    free(c->phi); free(c->phi_prev); free(c->dtphi); free(c->u); free(c->p); free(c->T); free(c->pdot);
    free(c->grad); free(c->lap); free(c->u_next); free(c->divuphi);
    free(c);
}

void oracle_set_cac_form(oracle_ctx *c, int form) { if (c) c->cac_form = form; }

/* Time-dependent prescribed velocity (reversing vortex: u'(x,t) = u(x) cos(pi t / 2 T_f)): the field
 * given here is u at the NEXT time level; the moments pass of the next step takes it as u^{n+1}.  The collision
 * of the next step still sees u^n, the field of the level it collides at. */
int oracle_set_velocity(oracle_ctx *c, const double *u)
{
    if (!c || !u || !(c->P.flags & ORA_PRESCRIBED_U)) return -1;
    if (!c->u_next) c->u_next = (double *)malloc(3 * (size_t)c->N * sizeof(double));
    if (!c->u_next) return -1;
    memcpy(c->u_next, u, 3 * (size_t)c->N * sizeof(double));
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * phi at a possibly out-of-domain position (reading S8-iv): the value a ghost layer filled axis by
 * axis (x, then y, then z) would hold.  Periodic axis: wrap.  Zero-flux face: mirror in the wall, which
 * sits half a cell outside the first node: phi(-1) = phi(0), phi(-2) = phi(1) (the second ghost layer is
 * reached by the second-order biased difference only).  Dirichlet face with value v:
 * phi(-1) = 2 v - phi(0), phi(-2) = 2 v - phi(1).
 * ---------------------------------------------------------------------------------------------- */
static double phi_at(const oracle_ctx *c, const double *phi, int x, int y, int z)
{
    int q[3] = { x, y, z };
    int kind[3] = { 0, 0, 0 };
    double val[3] = { 0, 0, 0 };
    for (int a = 0; a < 3; ++a) {
        int n = axis_len(c, a);
        if (q[a] >= 0 && q[a] < n) continue;
        int side = q[a] < 0 ? 0 : 1;
        if (c->P.bc_g[a][side] == ORA_S_PERIODIC) {
            q[a] = ((q[a] % n) + n) % n;
        } else {
            q[a] = side == 0 ? -1 - q[a] : 2 * n - 1 - q[a];
            kind[a] = c->P.bc_g[a][side];
            val[a] = c->P.bc_phi[a][side];
        }
    }
    double v = phi[idx(c, q[0], q[1], q[2])];
    for (int a = 0; a < 3; ++a)
        if (kind[a] == ORA_S_DIRICHLET) v = 2.0 * val[a] - v;
    return v;
}

/* P1 -- directional-derivative gradient and Laplacian, Eq.(35a,b) and (36a,b), PAPER.md:291-315,
 * on the NS lattice's directions with the printed factor 3 read as 1/e2 (reading S2).
 * The directional derivative inside Eq.(35b) is the central one, Eq.(35a), or one of the biased differences the paper
 * defines at PAPER.md:318; the Laplacian is Eq.(36a,b) in every case. */
static void pass_derive(oracle_ctx *c)
{
    const lattice_t *L = &c->Lf;
    const double dx = c->P.dx;
    const int nx = c->P.nx, ny = c->P.ny, nz = c->P.nz;
    const long N = c->N;
#pragma omp parallel for collapse(2)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double gx = 0, gy = 0, gz = 0, lp = 0;
                double ph0 = c->phi[idx(c, x, y, z)];
                for (int i = 1; i < L->Q; ++i) {
                    double php = phi_at(c, c->phi, x + L->e[i][0], y + L->e[i][1], z + L->e[i][2]);
                    double phm = phi_at(c, c->phi, x - L->e[i][0], y - L->e[i][1], z - L->e[i][2]);
                    double d1 = (php - phm) / (2.0 * dx);              /* Eq.(35a) */
                    if (c->P.grad_scheme == ORA_GRAD_BIASED1) {
                        d1 = (php - ph0) / dx;                         /* first-order biased */
                    } else if (c->P.grad_scheme == ORA_GRAD_BIASED2) { /* second-order biased */
                        double php2 = phi_at(c, c->phi, x + 2 * L->e[i][0], y + 2 * L->e[i][1], z + 2 * L->e[i][2]);
                        d1 = (-php2 + 4.0 * php - 3.0 * ph0) / (2.0 * dx);
                    }
                    double d2 = (php - 2.0 * ph0 + phm) / (dx * dx);   /* Eq.(36a) */
                    gx += L->w[i] * L->e[i][0] * d1;                   /* Eq.(35b) */
                    gy += L->w[i] * L->e[i][1] * d1;
                    gz += L->w[i] * L->e[i][2] * d1;
                    lp += L->w[i] * d2;                                /* Eq.(36b) */
                }
                long n = idx(c, x, y, z);
                c->grad[n] = gx / L->e2;
                c->grad[N + n] = gy / L->e2;
                c->grad[2 * N + n] = gz / L->e2;
                c->lap[n] = lp / L->e2;
            }
}

/* Velocity at a possibly out-of-domain position, for the stencil divergence (reading S17; the paper gives no rule).
 * Periodic axis: wrap.  No-slip wall half a cell outside the first node: odd reflection, u(-1) = -u(0), so that the
 * value interpolated on the wall is zero.  Open face: even reflection, u(-1) = u(0) (no normal gradient). */
static double u_at(const oracle_ctx *c, int comp, int x, int y, int z)
{
    int q[3] = { x, y, z };
    double sign = 1.0;
    for (int a = 0; a < 3; ++a) {
        int n = axis_len(c, a);
        if (q[a] >= 0 && q[a] < n) continue;
        int side = q[a] < 0 ? 0 : 1;
        if (c->P.bc_f[a][side] == ORA_F_PERIODIC) {
            q[a] = ((q[a] % n) + n) % n;
        } else {
            q[a] = side == 0 ? -1 - q[a] : 2 * n - 1 - q[a];
            if (c->P.bc_f[a][side] == ORA_F_WALL) sign = -sign;
        }
    }
    return sign * c->u[(long)comp * c->N + idx(c, q[0], q[1], q[2])];
}

/* ORA_DIV_STENCIL -- div(u phi) of Eq.(33d),(34) with the paper's own difference operator: each
 * d_a(u_a phi) by the directional derivatives Eq.(35a) assembled as in Eq.(35b), on the NS lattice,
 *   div(u phi) = (1/e2) sum_i w_i sum_a e_ia [ (u_a phi)(x + e_i) - (u_a phi)(x - e_i) ] / (2 dx),
 * from u and phi of the SAME level (reading S17).  The alternative to the product rule of reading S5. */
static void pass_divergence(oracle_ctx *c)
{
    const lattice_t *L = &c->Lf;
    const double dx = c->P.dx;
    const int nx = c->P.nx, ny = c->P.ny, nz = c->P.nz;
#pragma omp parallel for collapse(2)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                double d = 0.0;
                for (int i = 1; i < L->Q; ++i) {
                    int xp = x + L->e[i][0], yp = y + L->e[i][1], zp = z + L->e[i][2];
                    int xm = x - L->e[i][0], ym = y - L->e[i][1], zm = z - L->e[i][2];
                    double php = phi_at(c, c->phi, xp, yp, zp), phm = phi_at(c, c->phi, xm, ym, zm);
                    for (int a = 0; a < 3; ++a) {
                        if (!L->e[i][a]) continue;
                        double dd = (u_at(c, a, xp, yp, zp) * php - u_at(c, a, xm, ym, zm) * phm) / (2.0 * dx);
                        d += L->w[i] * L->e[i][a] * dd;
                    }
                }
                c->divuphi[idx(c, x, y, z)] = d / L->e2;
            }
}

/* Gamma_i, Eq.(27d), with the lattice's own w_i, c_i = e_i c, c_s^2 (reading S15). */
static double gamma_i(const lattice_t *L, int i, double cc, double cs2, const double u[3])
{
    double cu = cc * (L->e[i][0] * u[0] + L->e[i][1] * u[1] + L->e[i][2] * u[2]);
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    return L->w[i] * (1.0 + cu / cs2 + cu * cu / (2.0 * cs2 * cs2) - uu / (2.0 * cs2));
}

/* Eq.(18): Pdot = m'''/rho_g = -(4 alpha/(A W^2)) (theta_I - theta) phi (1 - phi),
 * theta = Cp (T - T_sat)/L; alpha(phi) linear between the phases (reading S6). */
static double production_rate(const oracle_ctx *c, double phi, double T)
{
    const oracle_params *P = &c->P;
    if (!(P->flags & ORA_PHASE_CHANGE)) return 0.0;
    double alpha = phi * P->alpha_g + (1.0 - phi) * P->alpha_l;
    double theta = P->Cp * (T - P->T_sat) / P->L_latent;
    return -(4.0 * alpha / (P->A * P->W * P->W)) * (P->theta_I - theta) * phi * (1.0 - phi);
}

/* Total force of Eq.(12) at one node from phi, grad phi, lap phi.
 * F_s = mu_phi grad phi, Eq.(13),(14) PAPER.md:114-118.
 * F_v = (rho - rho_l) g : buoyancy relative to the liquid, zero in pure liquid, pushes gas against g
 * (reading G6 of the printed F_v = (rho_l - rho) g).
 * A uniform body force (the paper replaces the pressure gradient of the Poiseuille tests by F = (G,0,0),
 * PAPER.md:418) is added to F_tot. */
static void total_force(const oracle_ctx *c, double phi, const double grad[3], double lap, double rho,
                        double F[3])
{
    const oracle_params *P = &c->P;
    double mu = 4.0 * c->H * phi * (phi - 1.0) * (phi - 0.5) - c->K * lap;
    for (int a = 0; a < 3; ++a) F[a] = mu * grad[a] + (rho - P->rho_l) * P->grav[a] + P->force[a];
}

/* P2 -- equilibria and sources of the three lattices at one node, from the level-n macros.
 * eq[k][i], S[k][i] with k = 0 (f), 1 (g), 2 (s); om[k] = 1/(tau_bar_k + 1/2). */
typedef struct { double eq[3][QMAX], S[3][QMAX], om[3]; } node_terms;

static void node_eq_sources(const oracle_ctx *c, long n, node_terms *t)
{
    const oracle_params *P = &c->P;
    const long N = c->N;
    const double dt = P->dt, cc = P->dx / P->dt;
    const double cs2f = c->Lf.e2 * cc * cc, cs2g = c->Lg.e2 * cc * cc, cs2s = c->Ls.e2 * cc * cc;
    const double drho = 1.0 / P->rho_g - 1.0 / P->rho_l;
    double phi = c->phi[n], T = c->T[n], p = c->p[n], dtphi = c->dtphi[n], pdot = c->pdot[n];
    double u[3] = { c->u[n], c->u[N + n], c->u[2 * N + n] };
    double grad[3] = { c->grad[n], c->grad[N + n], c->grad[2 * N + n] };
    double lap = c->lap[n];
    /* closures */
    double rho = phi * P->rho_g + (1.0 - phi) * P->rho_l;                        /* Eq.(1a) */
    double nu = P->nu_l * P->nu_g / (phi * P->nu_l + (1.0 - phi) * P->nu_g);     /* Eq.(1b) */
    double alpha = phi * P->alpha_g + (1.0 - phi) * P->alpha_l;                  /* reading S6 */
    double grho[3], F[3], nrm[3];
    for (int a = 0; a < 3; ++a) grho[a] = (P->rho_g - P->rho_l) * grad[a];       /* grad of Eq.(1a) */
    total_force(c, phi, grad, lap, rho, F);
    double gnorm = sqrt(grad[0] * grad[0] + grad[1] * grad[1] + grad[2] * grad[2] + P->eps_n * P->eps_n);
    for (int a = 0; a < 3; ++a) nrm[a] = grad[a] / gnorm;                        /* Eq.(6), reading S7 */
    double mdot = P->rho_g * pdot;                                               /* mass production rate */
    /* div(u phi) = u.grad phi + phi div u with div u = mdot (1/rho_g - 1/rho_l), Eq.(11a) (reading S5) */
    double D = u[0] * grad[0] + u[1] * grad[1] + u[2] * grad[2] + phi * mdot * drho;
    if (c->divuphi) D = c->divuphi[n];   /* ... or the stencil divergence of this level (reading S17) */
    /* relaxation rates: tau_bar = nu/(c_s^2 dt) PAPER.md:208, M/(c_s^2 dt) PAPER.md:236,
     * alpha/(c_s^2 dt) PAPER.md:272; om = 1/(tau_bar + 1/2), Eq.(25) */
    t->om[0] = 1.0 / (nu / (cs2f * dt) + 0.5);
    t->om[1] = 1.0 / (P->M / (cs2g * dt) + 0.5);
    t->om[2] = 1.0 / (alpha / (cs2s * dt) + 0.5);

    /* Navier-Stokes: f_eq Eq.(26b); S^f = F^f + P^f Eq.(27a-c) */
    for (int i = 0; i < c->Lf.Q; ++i) {
        const lattice_t *L = &c->Lf;
        double G = gamma_i(L, i, cc, cs2f, u);
        t->eq[0][i] = L->w[i] * p + rho * cs2f * (G - L->w[i]);
        double Fi = 0.0;
        for (int a = 0; a < 3; ++a)
            Fi += (cc * L->e[i][a] - u[a]) * ((G - L->w[i]) * grho[a] * cs2f + G * F[a]);   /* Eq.(27b) */
        double Pi = L->w[i] * rho * cs2f * mdot * drho;                                     /* Eq.(27c) */
        t->S[0][i] = Fi + Pi;
    }
    /* conservative Allen-Cahn */
    for (int i = 0; i < c->Lg.Q; ++i) {
        const lattice_t *L = &c->Lg;
        double G = gamma_i(L, i, cc, cs2g, u);
        double cn = cc * (L->e[i][0] * nrm[0] + L->e[i][1] * nrm[1] + L->e[i][2] * nrm[2]);
        if (c->cac_form == ORA_CAC_MODIFIED_EQ) {
            /* Eq.(31b) PAPER.md:251 and P_i^g of Eq.(30b) */
            t->eq[1][i] = phi * G + P->M * (4.0 / P->W) * phi * (1.0 - phi) * L->w[i] * cn / cs2g;
            t->S[1][i] = L->w[i] * pdot;
        } else {
            /* Eq.(29b) PAPER.md:234 and S^g = F^g + P^g, Eq.(30a,b) PAPER.md:238-242 */
            t->eq[1][i] = phi * G;
            t->S[1][i] = (4.0 / P->W) * phi * (1.0 - phi) * L->w[i] * cn + L->w[i] * pdot;
        }
    }
    /* heat: s_eq Eq.(33b); source Eq.(33c,d) with the sign of Eq.(34)/(11d) (reading G2) */
    for (int i = 0; i < c->Ls.Q; ++i) {
        const lattice_t *L = &c->Ls;
        double G = gamma_i(L, i, cc, cs2s, u);
        t->eq[2][i] = T * G;
        t->S[2][i] = 0.0;
        if (P->flags & ORA_LATENT_HEAT) t->S[2][i] = -L->w[i] * (P->L_latent / P->Cp) * (dtphi + D);
    }
}

/* P3 -- BGK collision, Eq.(25) PAPER.md:187 with theta_bar_eq = theta_eq - dt/2 S, Eq.(24) PAPER.md:182:
 * theta_bar* = theta_bar - om [theta_bar - theta_bar_eq] + dt S. */
static void pass_collide(oracle_ctx *c)
{
    const long N = c->N;
    const double dt = c->P.dt;
    const lattice_t *Ls[3] = { &c->Lf, &c->Lg, &c->Ls };
    double *in[3] = { c->f, c->g, c->s };
    double *out[3] = { c->fpost, c->gpost, c->spost };
#pragma omp parallel for
    for (long n = 0; n < N; ++n) {
        node_terms t;
        node_eq_sources(c, n, &t);
        for (int k = 0; k < 3; ++k)
            for (int i = 0; i < Ls[k]->Q; ++i) {
                double bar = in[k][(long)i * N + n];
                double bar_eq = t.eq[k][i] - 0.5 * dt * t.S[k][i];
                out[k][(long)i * N + n] = bar - t.om[k] * (bar - bar_eq) + dt * t.S[k][i];
            }
    }
}

/* P4 -- pull streaming of one distribution with boundary rules (readings S8-i,ii,v).
 * kind_of(axis, side) gives that distribution's rule; dirichlet value per face in val. */
static void stream_one(const oracle_ctx *c, const lattice_t *L, const double *post, double *out,
                       int is_f, const int bc[3][2], const double val[3][2])
{
    const int nx = c->P.nx, ny = c->P.ny, nz = c->P.nz;
    const long N = c->N;
#pragma omp parallel for collapse(2)
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                long n = idx(c, x, y, z);
                for (int i = 0; i < L->Q; ++i) {
                    int q[3] = { x - L->e[i][0], y - L->e[i][1], z - L->e[i][2] };
                    int hit_axis = -1, hit_side = 0;
                    for (int a = 0; a < 3; ++a) {
                        int len = axis_len(c, a);
                        if (q[a] >= 0 && q[a] < len) continue;
                        int side = q[a] < 0 ? 0 : 1;
                        if (bc[a][side] == 0) {           /* periodic (0 for both f and scalar kinds) */
                            q[a] = ((q[a] % len) + len) % len;
                        } else if (hit_axis < 0) {        /* lowest non-periodic axis decides */
                            hit_axis = a; hit_side = side;
                        }
                    }
                    double v;
                    if (hit_axis < 0) {
                        v = post[(long)i * N + idx(c, q[0], q[1], q[2])];
                    } else {
                        double back = post[(long)L->opp[i] * N + n]; /* same node, opposite direction */
                        int kind = bc[hit_axis][hit_side];
                        if (is_f) {
                            if (kind == ORA_F_WALL) v = back;
                            else v = -back + 2.0 * L->w[i] * val[hit_axis][hit_side];          /* S12: open */
                        } else {
                            if (kind == ORA_S_ZEROFLUX) v = back;
                            else v = -back + 2.0 * L->w[i] * val[hit_axis][hit_side];
                        }
                    }
                    out[(long)i * N + n] = v;
                }
            }
}

static void pass_stream(oracle_ctx *c)
{
    stream_one(c, &c->Lf, c->fpost, c->f, 1, c->P.bc_f, c->P.bc_p);
    stream_one(c, &c->Lg, c->gpost, c->g, 0, c->P.bc_g, c->P.bc_phi);
    stream_one(c, &c->Ls, c->spost, c->s, 0, c->P.bc_s, c->P.bc_T);
}

/* P5 -- moments at level n+1 in the order of reading S3. */
static void pass_moments(oracle_ctx *c)
{
    const oracle_params *P = &c->P;
    const long N = c->N;
    const double dt = P->dt, cc = P->dx / P->dt;
    const double cs2f = c->Lf.e2 * cc * cc;
    const double drho = 1.0 / P->rho_g - 1.0 / P->rho_l;
    /* 1,2: phi = sum g + dt/2 sum P_i^g with the stored Pdot (Eq.32); backward dphi/dt (S4) */
#pragma omp parallel for
    for (long n = 0; n < N; ++n) {
        double sum = 0.0;
        for (int i = 0; i < c->Lg.Q; ++i) sum += c->g[(long)i * N + n];
        double corr = 0.0;
        for (int i = 0; i < c->Lg.Q; ++i) corr += c->Lg.w[i] * c->pdot[n];
        double phinew = sum + 0.5 * dt * corr;
        c->phi_prev[n] = c->phi[n];
        c->dtphi[n] = (phinew - c->phi[n]) / dt;
        c->phi[n] = phinew;
    }
    /* 3: derived fields of the new phi */
    pass_derive(c);
    /* 4: rho u = (1/c_s^2) sum f c_i + dt/2 F_tot, Eq.(28a) PAPER.md:224 -- for every node before any of 5-8, because the
     * stencil divergence (ORA_DIV_STENCIL) reads the neighbours' new velocity */
#pragma omp parallel for
    for (long n = 0; n < N; ++n) {
        double phi = c->phi[n];
        double grad[3] = { c->grad[n], c->grad[N + n], c->grad[2 * N + n] };
        double rho = phi * P->rho_g + (1.0 - phi) * P->rho_l;
        double F[3], u[3];
        total_force(c, phi, grad, c->lap[n], rho, F);
        double m1[3] = { 0, 0, 0 };
        for (int i = 0; i < c->Lf.Q; ++i) {
            double fi = c->f[(long)i * N + n];
            for (int a = 0; a < 3; ++a) m1[a] += fi * cc * c->Lf.e[i][a];
        }
        for (int a = 0; a < 3; ++a) u[a] = (m1[a] / cs2f + 0.5 * dt * F[a]) / rho;
        /* prescribed-velocity verifications (Zalesak disk, vortex): u stays the given field */
        if (P->flags & ORA_PRESCRIBED_U) {
            const double *up = c->u_next ? c->u_next : c->u;   /* u(x, t^{n+1}) */
            for (int a = 0; a < 3; ++a) u[a] = up[(long)a * N + n];
        }
        for (int a = 0; a < 3; ++a) c->u[(long)a * N + n] = u[a];
    }
    if (c->divuphi) pass_divergence(c);   /* div(u^{n+1} phi^{n+1}) by the stencil (reading S17) */
    /* 5-8 */
#pragma omp parallel for
    for (long n = 0; n < N; ++n) {
        double phi = c->phi[n];
        double grad[3] = { c->grad[n], c->grad[N + n], c->grad[2 * N + n] };
        double rho = phi * P->rho_g + (1.0 - phi) * P->rho_l;
        double grho[3], u[3];
        for (int a = 0; a < 3; ++a) grho[a] = (P->rho_g - P->rho_l) * grad[a];
        for (int a = 0; a < 3; ++a) u[a] = c->u[(long)a * N + n];
        double m0 = 0.0;
        for (int i = 0; i < c->Lf.Q; ++i) m0 += c->f[(long)i * N + n];
        /* 5: m''' from the stored Pdot; D = div(u phi) (S5) */
        double mdot = P->rho_g * c->pdot[n];
        double D = u[0] * grad[0] + u[1] * grad[1] + u[2] * grad[2] + phi * mdot * drho;
        if (c->divuphi) D = c->divuphi[n];
        /* 6: T = sum s - dt/2 (L/Cp) [dphi/dt + div(u phi)], Eq.(34) */
        double T = 0.0;
        for (int i = 0; i < c->Ls.Q; ++i) T += c->s[(long)i * N + n];
        if (P->flags & ORA_LATENT_HEAT) T -= 0.5 * dt * (P->L_latent / P->Cp) * (c->dtphi[n] + D);
        /* 7: p = sum f + dt/2 { c_s^2 u.grad rho + rho c_s^2 m''' (1/rho_g - 1/rho_l) }, Eq.(28b) */
        double ugr = u[0] * grho[0] + u[1] * grho[1] + u[2] * grho[2];
        double p = m0 + 0.5 * dt * (cs2f * ugr + rho * cs2f * mdot * drho);
        c->T[n] = T;
        c->p[n] = p;
        /* 8: refresh the production field with the new macros, Eq.(18) */
        c->pdot[n] = production_rate(c, phi, T);
    }
}

/* Initialisation (reading S9; the paper gives none): dphi/dt = 0, Pdot from the initial macros (Eq.18),
 * populations at bar-equilibrium, theta_bar = theta_eq - dt/2 S (Eq.24), so that the
 * moment formulas (28a,b), (32), (34) return the initial macros. */
int oracle_init(oracle_ctx *c, const double *phi, const double *T, const double *u, const double *p)
{
    if (!c || !phi) return -1;
    const oracle_params *P = &c->P;
    const long N = c->N;
    for (long n = 0; n < N; ++n) {
        c->phi[n] = phi[n];
        c->phi_prev[n] = phi[n];
        c->dtphi[n] = 0.0;
        c->T[n] = T ? T[n] : P->T_sat;
        c->p[n] = p ? p[n] : 0.0;
        for (int a = 0; a < 3; ++a) c->u[(long)a * N + n] = u ? u[(long)a * N + n] : 0.0;
        c->pdot[n] = production_rate(c, c->phi[n], c->T[n]);
    }
    c->nsteps = 0;
    pass_derive(c);
    if (c->divuphi) pass_divergence(c);
    const lattice_t *Ls[3] = { &c->Lf, &c->Lg, &c->Ls };
    double *pops[3] = { c->f, c->g, c->s };
#pragma omp parallel for
    for (long n = 0; n < N; ++n) {
        node_terms t;
        node_eq_sources(c, n, &t);
        for (int k = 0; k < 3; ++k)
            for (int i = 0; i < Ls[k]->Q; ++i)
                pops[k][(long)i * N + n] = t.eq[k][i] - 0.5 * P->dt * t.S[k][i];
    }
    return 0;
}

int oracle_step(oracle_ctx *c, int nsteps)
{
    if (!c || nsteps < 0) return -1;
    for (int k = 0; k < nsteps; ++k) {
        /* P1: grad phi, lap phi of level n are already in place -- oracle_init and pass_moments end with
         * pass_derive on the same phi */
        pass_collide(c);  /* P2, P3 */
        pass_stream(c);   /* P4 */
        pass_moments(c);  /* P5 */
        c->nsteps++;
    }
    return 0;
}

int oracle_read_macro(oracle_ctx *c, double *phi, double *u, double *p, double *T)
{
    if (!c) return -1;
    const long N = c->N;
    if (phi) memcpy(phi, c->phi, N * sizeof(double));
    if (u) memcpy(u, c->u, 3 * N * sizeof(double));
    if (p) memcpy(p, c->p, N * sizeof(double));
    if (T) memcpy(T, c->T, N * sizeof(double));
    return 0;
}

int oracle_read_pops(oracle_ctx *c, int which, int stage, double *out)
{
    if (!c || !out || which < 0 || which > 2) return -1;
    const lattice_t *L = which == 0 ? &c->Lf : (which == 1 ? &c->Lg : &c->Ls);
    const double *src;
    if (stage == ORA_POPS_STREAMED) {
        src = which == 0 ? c->f : (which == 1 ? c->g : c->s);
    } else {
        pass_derive(c);
        pass_collide(c); /* post-collision populations of the current level; state is not advanced */
        src = which == 0 ? c->fpost : (which == 1 ? c->gpost : c->spost);
    }
    memcpy(out, src, (size_t)L->Q * c->N * sizeof(double));
    return 0;
}

int oracle_read_div(oracle_ctx *c, double *div)
{
    if (!c || !div || !c->divuphi) return -1;
    memcpy(div, c->divuphi, (size_t)c->N * sizeof(double));
    return 0;
}

int oracle_read_aux(oracle_ctx *c, double *grad, double *lap, double *pdot, double *dtphi)
{
    if (!c) return -1;
    const long N = c->N;
    pass_derive(c);
    if (grad) memcpy(grad, c->grad, 3 * N * sizeof(double));
    if (lap) memcpy(lap, c->lap, N * sizeof(double));
    if (pdot) memcpy(pdot, c->pdot, N * sizeof(double));
    if (dtphi) memcpy(dtphi, c->dtphi, N * sizeof(double));
    return 0;
}
