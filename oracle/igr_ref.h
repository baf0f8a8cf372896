/* igr_ref.h -- fp64 CPU ORACLE for one SSP-RK3 step of the 3D compressible Euler
 * equations with information geometric regularisation (IGR).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, step-by-step
 * restatement of the discretisation of arXiv 2505.07392, written from the
 * paper and SURVEY.md section 8(c) only.  It shares no code, header, table or helper
 * with the CUDA path (paper_2505_07392_b200/csrc, include/igr.h).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load it.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): reconstruction exactness on
 * monomials (P1), fifth-difference dissipation (P2), LF consistency (P3), RK3 order
 * (P4), source on linear velocity fields (P5), Jacobi vs dense solve / contraction
 * 60/61 (P6), uniform state bitwise (P7), conservation (P8), scale covariance (P9),
 * entropy-wave convergence order (P10), Sod vs exact Riemann solution (P11), axis
 * permutation symmetry (P12), periodic-doubling and inflow mask (P13); viscous fluxes
 * (NEXT-1): textbook stress cases, tau:grad u heating, discrete shear-wave decay (P14);
 * the CFL wave speed against its closed form (P15); the cell-centred sound speed and the
 * local LF speed inside igr_ref_rhs against the textbook Rusanov flux worked out by hand
 * beside a density jump (P16).  tests/test_oracle_f1.py records what the scheme as read
 * does on the inputs as BASELINE.json states them (finding F1).
 * Parity unpinned by any external value (fixed by DESIGN.md readings A2-A5 only):
 * the 5-sweep truncation, the warm-start order, the CHOICE of the local cell-centred LF
 * speed (its formula is pinned by P16) and the arithmetic-mean face density.
 *
 * Layout: every field is a padded array [nz+2*NG][ny+2*NG][nx+2*NG], x fastest,
 * NG = 3 ghost layers on every side.  State q = (rho, m_x, m_y, m_z, E).
 */
#ifndef IGR_REF_H
#define IGR_REF_H

#ifdef __cplusplus
extern "C" {
#endif

#define IGR_REF_NG 3

/* face codes */
#define IGR_REF_BC_PERIODIC 0
#define IGR_REF_BC_EXTRAP   1
#define IGR_REF_BC_INFLOW   2
/* face shared with a neighbouring sub-domain (domain decomposition; DESIGN.md reading
 * A20): ghosts beyond it are never filled by the oracle, the caller provides them (set_padded)    */
#define IGR_REF_BC_EXTERNAL 3

/* storage emulation ("FP32 compute, FP16 storage") */
#define IGR_REF_STORE_F64  0
#define IGR_REF_STORE_F32  1
#define IGR_REF_STORE_F16  2
#define IGR_REF_STORE_BF16 3

typedef struct {
    double c0, c1, radius;      /* centre and radius in CELL units on the face plane;   */
                                /* transverse axes in the order x<y<z                    */
    double edge;                /* 0: sharp mask r <= radius; > 0: tanh edge of this     */
                                /* half-width (cells), reading A8b                       */
    double rho, u, v, w, p;     /* fixed primitive state                                 */
} igr_ref_patch;

typedef struct {
    int face[6];                /* x-,x+,y-,y+,z-,z+                                     */
    int n_patches[6];
    const igr_ref_patch *patches[6];
} igr_ref_bc;

typedef struct igr_ref_solver igr_ref_solver;

int  igr_ref_create(int nx, int ny, int nz, double dx, double gamma, double alpha,
                    int order, int n_jacobi, const igr_ref_bc *bc, igr_ref_solver **out);
void igr_ref_destroy(igr_ref_solver *s);
int  igr_ref_set_storage(igr_ref_solver *s, int mode);       /* IGR_REF_STORE_*         */
/* NEXT-1: shear and bulk viscosity of eq. (5) (L64-L67); 0, 0 = inviscid Euler (default) */
int  igr_ref_set_viscosity(igr_ref_solver *s, double mu, double zeta);

/* interior-only host arrays, layout [5][nz][ny][nx] (state) or [nz][ny][nx] (scalar) */
int  igr_ref_set_state(igr_ref_solver *s, const double *q);  /* also resets Sigma = 0   */
int  igr_ref_get_state(const igr_ref_solver *s, double *q);
int  igr_ref_set_sigma(igr_ref_solver *s, const double *sig);
int  igr_ref_get_sigma(const igr_ref_solver *s, double *sig);
int  igr_ref_get_source(const igr_ref_solver *s, double *b); /* last computed b         */
int  igr_ref_set_source(igr_ref_solver *s, const double *b); /* test hook for the sweeps */
int  igr_ref_get_rhs(const igr_ref_solver *s, double *r);    /* last computed r [5]...  */
/* padded copy of q component c (0..4) or Sigma (c = 5): [nz+6][ny+6][nx+6]            */
int  igr_ref_get_padded(const igr_ref_solver *s, int c, double *out);
int  igr_ref_set_padded(igr_ref_solver *s, int c, const double *in);   /* inverse of get_padded */

int  igr_ref_max_wavespeed(const igr_ref_solver *s, double *out);
int  igr_ref_step(igr_ref_solver *s, double dt);             /* one SSP-RK3 step        */
int  igr_ref_stage(igr_ref_solver *s, int stage, double dt); /* stage 1, 2, 3 of that step */

/* the pieces of one RHS evaluation L(q, Sigma_prev) -> (r, Sigma), in order           */
int  igr_ref_fill_ghosts(igr_ref_solver *s);   /* step 1: ghosts of q + primitives      */
int  igr_ref_source(igr_ref_solver *s);        /* step 2: b                             */
int  igr_ref_jacobi_sweep(igr_ref_solver *s);  /* step 3: refresh Sigma ghosts, 1 sweep */
int  igr_ref_solve_sigma(igr_ref_solver *s);   /* step 3: n_jacobi sweeps + ghosts      */
int  igr_ref_fill_sigma_ghosts(igr_ref_solver *s);
int  igr_ref_rhs(igr_ref_solver *s);           /* steps 4-7: r from q, Sigma            */
int  igr_ref_eval_rhs(igr_ref_solver *s);      /* steps 1-7                             */

/* stand-alone array helpers used by the pins */
/* out = a*qn + b*(qs + dt*r), elementwise over n values (SSP-RK3 stage combination)   */
void igr_ref_rk_combine(double a, const double *qn, double b, const double *qs,
                        double dt, const double *r, double *out, long n);
/* left/right face values at the face between cells 0 and 1 from cells -2..3 (f[0..5]) */
void igr_ref_reconstruct(int order, const double *f6, double *fL, double *fR);
/* LF flux along axis d from reconstructed conservative L/R states (5 values each),    */
/* Sigma_L, Sigma_R and the wave speed lambda                                          */
void igr_ref_lf_flux(int d, double gamma, const double *UL, const double *UR,
                     double sigL, double sigR, double lambda, double *F);
/* viscous flux along d from face values of G[3a+b] = du_a/dx_b and of the velocity   */
void igr_ref_viscous_flux(int d, double mu, double zeta, const double *G9, const double *u3, double *F);
/* round x to the storage format (round to nearest even)                               */
double igr_ref_round_storage(double x, int mode);

/* ---------------------------------------------------------------- two-fluid variant (NEXT-3)
 * igr_ref2.c: five-equation (volume-fraction) model of two ideal gases, reading A21; see the header of that
 * file for the passages of the paper it follows and for its pins.  State layout [7][nz][ny][nx]:
 * (a1 rho1, a2 rho2, rho u, rho v, rho w, E, a1). */
typedef struct {
    double c0, c1, radius, edge;          /* as igr_ref_patch                                  */
    double a1rho1, a2rho2, a1;            /* partial densities and volume fraction of fluid 1  */
    double u, v, w, p;
} igr_ref2_patch;

typedef struct {
    int face[6];                          /* periodic / extrapolation / inflow                 */
    int n_patches[6];
    const igr_ref2_patch *patches[6];
} igr_ref2_bc;

typedef struct igr_ref2_solver igr_ref2_solver;

int  igr_ref2_create(int nx, int ny, int nz, double dx, double gamma1, double gamma2, double alpha, int order,
                     int n_jacobi, const igr_ref2_bc *bc, igr_ref2_solver **out);
void igr_ref2_destroy(igr_ref2_solver *s);
int  igr_ref2_set_state(igr_ref2_solver *s, const double *q);     /* also resets Sigma = 0 */
int  igr_ref2_get_state(const igr_ref2_solver *s, double *q);
int  igr_ref2_get_rhs(const igr_ref2_solver *s, double *r);       /* last computed r [7]... */
int  igr_ref2_get_sigma(const igr_ref2_solver *s, double *sig);
int  igr_ref2_set_sigma(igr_ref2_solver *s, const double *sig);
int  igr_ref2_get_source(const igr_ref2_solver *s, double *b);
int  igr_ref2_get_padded(const igr_ref2_solver *s, int c, double *out);   /* c = 0..6, 7 = Sigma */
int  igr_ref2_max_wavespeed(const igr_ref2_solver *s, double *out);
int  igr_ref2_step(igr_ref2_solver *s, double dt);
int  igr_ref2_stage(igr_ref2_solver *s, int stage, double dt);
int  igr_ref2_fill_ghosts(igr_ref2_solver *s);
int  igr_ref2_source(igr_ref2_solver *s);
int  igr_ref2_solve_sigma(igr_ref2_solver *s);
int  igr_ref2_rhs(igr_ref2_solver *s);
int  igr_ref2_eval_rhs(igr_ref2_solver *s);

#ifdef __cplusplus
}
#endif
#endif
