/*
 * CPU ORACLE -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision restatement of the coupled phase-field lattice Boltzmann step of
 * Verdier, Kestener, Cartalade, "Performance portability of lattice Boltzmann methods for two-phase
 * flows with phase change", following the paper's equations pass by pass (separate
 * derive / collide / stream / moment loops, no fusion, no blocking).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use
 * anything under oracle/.  The product (paper_2003_06342_b200/) never includes, links or imports it,
 * and this directory shares no header, table or helper with the CUDA path.
 *
 * Readings of garbled / silent passages of the paper are the ones listed in DESIGN.md ("Readings");
 * tags G* / S* in comments refer to that list.
 *
 * Parity unpinned: nothing outright; two READINGS the paper cannot confirm stay readings.
 * div(u phi): the paper does not say how it discretised it.  Both candidates are here and both are pinned: the product rule of
 * reading S5 (u.grad(phi) by Galilean invariance of the latent-heat source, phi div u by the Eq.(11a) mass balance) and the
 * stencil divergence of reading S17 (equal to u.grad(phi) for uniform u, exact on quadratic fluxes, wall / open ghost rule);
 * which of the two the paper's authors ran is what stays open.
 * The OPEN pressure face (S12, not in the paper) is pinned in the role config 2 gives it -- normal outflow at a fixed
 * pressure: exact hydrostatic column, outflow = integrated mass source; its behaviour under shear is not (a 32 x 16
 * pressure-driven channel carries 6.5 % more flux than Poiseuille's law, entry effect of the plain anti-bounce-back).
 * The 3D coupling terms (not run in 3D by the paper) are pinned by the spherical Laplace law,
 * the symmetry tests and the brute-force comparison; everything else by tests/test_oracle_*.py.
 */
#ifndef LBM_ORACLE_H
#define LBM_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* lattice ids (D2Q5 is not in the paper, reading S1) */
enum { ORA_D2Q5 = 0, ORA_D2Q9 = 1, ORA_D3Q7 = 2, ORA_D3Q19 = 3, ORA_D3Q15 = 4 };
/* boundary kinds of the Navier-Stokes distribution f, per face */
enum { ORA_F_PERIODIC = 0, ORA_F_WALL = 1 /* half bounce-back */,
       ORA_F_OPEN = 2 /* pressure anti-bounce-back, reading S12 */ };
/* boundary kinds of the scalar distributions g (phase field) and s (temperature), per face */
enum { ORA_S_PERIODIC = 0, ORA_S_ZEROFLUX = 1 /* bounce-back */,
       ORA_S_DIRICHLET = 2 /* anti-bounce-back */ };
/* flags */
enum { ORA_PHASE_CHANGE = 1u /* Eq.(18) production rate on */,
       ORA_LATENT_HEAT = 2u /* Eq.(33c,d),(34) source of the heat equation on */,
       ORA_PRESCRIBED_U = 4u /* u is the field given to oracle_init and is not updated from f */ };
/* conservative Allen-Cahn collision form */
enum { ORA_CAC_MODIFIED_EQ = 0 /* Eq.(31a,b) */, ORA_CAC_SOURCE = 1 /* Eq.(29a,b),(30a,b) */ };
/* directional derivative e_i.grad(phi) used in the gradient Eq.(35b): central Eq.(35a), or the biased differences of
 * first order [phi(x+e) - phi(x)]/dx, second order [-phi(x+2e) + 4 phi(x+e) - 3 phi(x)]/(2 dx) */
enum { ORA_GRAD_CENTRAL = 0, ORA_GRAD_BIASED1 = 1, ORA_GRAD_BIASED2 = 2 };
/* div(u phi) of Eq.(33d),(34): product rule u.grad(phi) + phi div u with Eq.(11a) (reading S5), or the directional-derivative
 * stencil Eq.(35a,b) applied to the components of u phi (reading S17) */
enum { ORA_DIV_PRODUCT = 0, ORA_DIV_STENCIL = 1 };
/* stage selector of oracle_read_pops */
enum { ORA_POPS_POSTCOLLISION = 0, ORA_POPS_STREAMED = 1 };

typedef struct oracle_params {
    int nx, ny, nz;               /* nz == 1 : two-dimensional                                   */
    int lat_f, lat_g, lat_s;      /* lattice of f (NS), g (Allen-Cahn), s (heat)                 */
    int bc_f[3][2];               /* [axis][lo,hi]                                               */
    int bc_g[3][2];
    int bc_s[3][2];
    double bc_phi[3][2];          /* Dirichlet values of phi                                     */
    double bc_T[3][2];            /* Dirichlet values of T                                       */
    double bc_p[3][2];            /* pressure of OPEN faces                                      */
    double dx, dt;
    double rho_l, rho_g, nu_l, nu_g;
    double sigma, W, M;           /* surface tension, interface width, mobility                  */
    double grav[3];               /* gravity acceleration vector g (points "down")               */
    double force[3];              /* uniform body force density added to F_tot    */
    double alpha_l, alpha_g;      /* thermal diffusivities                                       */
    double L_latent, Cp, T_sat, theta_I;
    double A;                     /* script-A of Eq.(18); 10/48 in the paper      */
    double eps_n;                 /* regularisation of n = grad phi / |grad phi| (reading S7)    */
    unsigned flags;
    int grad_scheme;              /* ORA_GRAD_*: directional derivative inside Eq.(35b) */
    int div_scheme;               /* ORA_DIV_*: discretisation of div(u phi)                          */
} oracle_params;

typedef struct oracle_ctx oracle_ctx;

/* returns NULL on invalid parameters */
oracle_ctx *oracle_create(const oracle_params *p);
void oracle_destroy(oracle_ctx *c);
/* arrays are x-fastest [z][y][x]; u is [comp][z][y][x] with 3 components; NULL => u=0, p=0, T=T_sat */
int oracle_init(oracle_ctx *c, const double *phi, const double *T, const double *u, const double *p);
int oracle_step(oracle_ctx *c, int n);
int oracle_read_macro(oracle_ctx *c, double *phi, double *u, double *p, double *T);
/* which: 0=f, 1=g, 2=s ; out is [Q][z][y][x] */
int oracle_read_pops(oracle_ctx *c, int which, int stage, double *out);
/* auxiliary fields for the pins: grad phi [3][N], laplacian [N], production rate Pdot [N], dphi/dt [N] */
int oracle_read_aux(oracle_ctx *c, double *grad, double *lap, double *pdot, double *dtphi);
/* ORA_DIV_STENCIL only: the stencil divergence of (u phi) at the current level [N] */
int oracle_read_div(oracle_ctx *c, double *div);
void oracle_set_cac_form(oracle_ctx *c, int form);
/* ORA_PRESCRIBED_U only: u [3][z][y][x] of the next time level (time-dependent prescribed velocity) */
int oracle_set_velocity(oracle_ctx *c, const double *u);
int oracle_num_threads(void);
/* lattice table access for the pins: returns Q, fills e[Q][3], w[Q], *e2 */
int oracle_lattice(int id, int *e, double *w, double *e2);

#ifdef __cplusplus
}
#endif
#endif
