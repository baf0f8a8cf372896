/* igr_ref2.c -- fp64 CPU ORACLE of the TWO-FLUID variant (test infrastructure, not the product).
 *
 * the workload behind every number of the paper's Table 1 and
 * both scaling figures (L297) is a two-fluid problem.  The paper gives no equations for it; what it does give:
 *   - Alg. 1: the conservative variables are (rho, rho u, E, alpha): the volume fraction alpha (NOT the
 *     IGR alpha) is carried as one more conserved/advected block and updated like the others (L228);
 *   - L196: alpha_L, alpha_R <- alpha(-2:3) along idir: it is reconstructed with the same stencil;
 *   - L187-L198: the RECONSTRUCTED conservative variables are converted to primitives at the face;
 *   - L210: flux(rho_d, u_d, E_d, p_d, alpha_d, sigma_d): alpha enters the flux routine;
 *   - L363: "one- and two-fluid (or species) cases"; the code base is MFC (refs 7, 13, 32: the five-equation
 *     model of multicomponent flow).
 * Reading A21 takes the simplest closure consistent with this: two ideal gases (gamma_1, gamma_2) in
 * the five-equation (volume-fraction) model,
 *   q = (a1 rho1, a2 rho2, rho u, rho v, rho w, E, a1),   rho = a1 rho1 + a2 rho2,   a2 = 1 - a1,
 *   d(ai rhoi)/dt + div(ai rhoi u)                 = 0            (each partial mass is conserved)
 *   d(rho u)/dt  + div(rho u u + (p + Sigma) I)    = 0            (eq. 7)
 *   dE/dt        + div((E + p + Sigma) u)          = 0            (eq. 8)
 *   da1/dt       + div(a1 u) = a1 div u                            (advection, quasi-conservative form)
 *   p = (E - rho |u|^2 / 2) / Gamma,  Gamma = a1/(gamma_1 - 1) + a2/(gamma_2 - 1)   (isobaric mixture rule)
 *   c^2 = (1 + 1/Gamma) p / rho,  Sigma from eq. (9) with the mixture density.
 * Discretisation exactly as the single-fluid oracle (igr_ref.c): ghosts by the BC index map,
 * second-order source, n_jacobi warm-started sweeps, fifth-order linear reconstruction of the SEVEN conservative
 * fields and Sigma, primitives from the reconstructed values, local Lax-Friedrichs flux with the cell-centred
 * speed of the two adjacent cells, SSP-RK3.  Two details that the five-equation model needs:
 *   - the partial mass fluxes are written Y_i m_d with Y_i = (ai rhoi)/rho (identical to ai rhoi u_d; in the
 *     single-fluid limit it is m_d bitwise, the flux of igr_ref.c);
 *   - the term a1 div u uses the cell value of a1 and the face velocities u^ = (u_d,L + u_d,R)/2 of the same
 *     reconstruction: r_a = - sum_d (F^a_{i+1/2} - F^a_{i-1/2})/dx + a1_i sum_d (u^_{i+1/2} - u^_{i-1/2})/dx.
 *     With it a uniform velocity and pressure stay uniform across a material interface to round-off.
 * Pins (tests/test_oracle_twofluid.py): single-fluid limit against igr_ref.c (bitwise with gamma = 1.5, to
 * round-off with 1.4); uniform u, p preserved across an advected interface (fails for a linearly mixed gamma);
 * conservation of each partial mass, of momentum and of energy; a1 stays uniform in a uniform dilatation (the
 * non-conservative term); the mixture wave speed against its closed form.
 * Parity unpinned by any external value: the choice of this closure and of u^ (reading A21).
 *
 * It uses three pinned pieces of igr_ref.c as library steps: igr_ref_reconstruct (P1), igr_ref_rk_combine (P4),
 * and the patch / index-map conventions restated below. */
#include "igr_ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NG IGR_REF_NG
#define NF 7                      /* a1 rho1, a2 rho2, m_x, m_y, m_z, E, a1 */

struct igr_ref2_solver {
    int nx, ny, nz;
    long sx, sy, sz, np;
    double dx, gamma1, gamma2, alpha;
    int order, n_jacobi;
    int face[6];
    int n_patches[6];
    igr_ref2_patch *patches[6];
    double *q[NF], *qn[NF], *r[NF], *flux[NF];
    double *uhat;                 /* face velocity u^ of one axis, stored at the left cell */
    double *rho, *u[3], *p, *c;   /* cell-centred mixture density and primitives incl. ghosts */
    double *sig, *sig2, *b;
};

static long IDX(const igr_ref2_solver *s, int i, int j, int k)
{
    return (long)(i + NG) + s->sy * (long)(j + NG) + s->sz * (long)(k + NG);
}

static double big_gamma(const igr_ref2_solver *s, double a1)
{
    return a1 / (s->gamma1 - 1.0) + (1.0 - a1) / (s->gamma2 - 1.0);
}

int igr_ref2_create(int nx, int ny, int nz, double dx, double gamma1, double gamma2, double alpha, int order,
                    int n_jacobi, const igr_ref2_bc *bc, igr_ref2_solver **out)
{
    if (!out || !bc || nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(gamma1 > 1) || !(gamma2 > 1) || alpha < 0 ||
        n_jacobi < 0 || (order != 5 && order != 3))
        return -1;
    for (int a = 0; a < 3; ++a) {
        int lo = bc->face[2 * a], hi = bc->face[2 * a + 1];
        if ((lo == IGR_REF_BC_PERIODIC) != (hi == IGR_REF_BC_PERIODIC)) return -2;
        if (lo < 0 || lo > 2 || hi < 0 || hi > 2) return -2;
    }
    igr_ref2_solver *s = (igr_ref2_solver *)calloc(1, sizeof(*s));
    if (!s) return -3;
    s->nx = nx; s->ny = ny; s->nz = nz;
    s->sx = 1; s->sy = nx + 2 * NG; s->sz = s->sy * (ny + 2 * NG);
    s->np = s->sz * (nz + 2 * NG);
    s->dx = dx; s->gamma1 = gamma1; s->gamma2 = gamma2; s->alpha = alpha;
    s->order = order; s->n_jacobi = n_jacobi;
    for (int f = 0; f < 6; ++f) {
        s->face[f] = bc->face[f];
        s->n_patches[f] = (bc->face[f] == IGR_REF_BC_INFLOW) ? bc->n_patches[f] : 0;
        if (s->n_patches[f] > 0) {
            s->patches[f] = (igr_ref2_patch *)malloc(sizeof(igr_ref2_patch) * s->n_patches[f]);
            memcpy(s->patches[f], bc->patches[f], sizeof(igr_ref2_patch) * s->n_patches[f]);
        }
    }
    for (int c = 0; c < NF; ++c) {
        s->q[c] = (double *)calloc(s->np, sizeof(double)); s->qn[c] = (double *)calloc(s->np, sizeof(double));
        s->r[c] = (double *)calloc(s->np, sizeof(double)); s->flux[c] = (double *)calloc(s->np, sizeof(double));
    }
    s->uhat = (double *)calloc(s->np, sizeof(double));
    s->rho = (double *)calloc(s->np, sizeof(double));
    for (int a = 0; a < 3; ++a) s->u[a] = (double *)calloc(s->np, sizeof(double));
    s->p = (double *)calloc(s->np, sizeof(double)); s->c = (double *)calloc(s->np, sizeof(double));
    s->sig = (double *)calloc(s->np, sizeof(double)); s->sig2 = (double *)calloc(s->np, sizeof(double));
    s->b = (double *)calloc(s->np, sizeof(double));
    *out = s;
    return 0;
}

void igr_ref2_destroy(igr_ref2_solver *s)
{
    if (!s) return;
    for (int c = 0; c < NF; ++c) { free(s->q[c]); free(s->qn[c]); free(s->r[c]); free(s->flux[c]); }
    free(s->uhat); free(s->rho);
    for (int a = 0; a < 3; ++a) free(s->u[a]);
    free(s->p); free(s->c); free(s->sig); free(s->sig2); free(s->b);
    for (int f = 0; f < 6; ++f) free(s->patches[f]);
    free(s);
}

/* ---------------------------------------------------------------- interior copies */
static void put_interior(const igr_ref2_solver *s, double *dst, const double *src)
{
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) dst[IDX(s, i, j, k)] = src[((long)k * s->ny + j) * s->nx + i];
}

static void take_interior(const igr_ref2_solver *s, const double *src, double *dst)
{
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) dst[((long)k * s->ny + j) * s->nx + i] = src[IDX(s, i, j, k)];
}

int igr_ref2_set_state(igr_ref2_solver *s, const double *q)
{
    if (!s || !q) return -1;
    long n = (long)s->nx * s->ny * s->nz;
    for (int c = 0; c < NF; ++c) put_interior(s, s->q[c], q + c * n);
    memset(s->sig, 0, sizeof(double) * s->np);            /* "Sigma = 0 at t = 0" */
    memset(s->sig2, 0, sizeof(double) * s->np);
    return 0;
}

int igr_ref2_get_state(const igr_ref2_solver *s, double *q)
{
    if (!s || !q) return -1;
    long n = (long)s->nx * s->ny * s->nz;
    for (int c = 0; c < NF; ++c) take_interior(s, s->q[c], q + c * n);
    return 0;
}

int igr_ref2_get_rhs(const igr_ref2_solver *s, double *r)
{
    if (!s || !r) return -1;
    long n = (long)s->nx * s->ny * s->nz;
    for (int c = 0; c < NF; ++c) take_interior(s, s->r[c], r + c * n);
    return 0;
}

int igr_ref2_get_sigma(const igr_ref2_solver *s, double *sig)
{
    if (!s || !sig) return -1;
    take_interior(s, s->sig, sig);
    return 0;
}

int igr_ref2_set_sigma(igr_ref2_solver *s, const double *sig)
{
    if (!s || !sig) return -1;
    put_interior(s, s->sig, sig);
    return 0;
}

int igr_ref2_get_source(const igr_ref2_solver *s, double *b)
{
    if (!s || !b) return -1;
    take_interior(s, s->b, b);
    return 0;
}

int igr_ref2_get_padded(const igr_ref2_solver *s, int c, double *out)
{
    if (!s || !out || c < 0 || c > NF) return -1;
    memcpy(out, c < NF ? s->q[c] : s->sig, sizeof(double) * s->np);
    return 0;
}

/* ---------------------------------------------------------------- boundary conditions (as igr_ref.c) */
static int map_index(int i, int n, int face_lo)
{
    if (i >= 0 && i < n) return i;
    if (face_lo == IGR_REF_BC_PERIODIC) { int m = i % n; return m < 0 ? m + n : m; }
    return i < 0 ? 0 : n - 1;
}

static double patch_weight(const igr_ref2_patch *pt, int t0, int t1)
{
    double d0 = (t0 + 0.5) - pt->c0, d1 = (t1 + 0.5) - pt->c1;
    double r2 = d0 * d0 + d1 * d1;
    if (pt->edge <= 0.0) return (r2 <= pt->radius * pt->radius) ? 1.0 : 0.0;
    double r = sqrt(r2);
    if (r >= pt->radius + 4.0 * pt->edge) return 0.0;
    return 0.5 * (1.0 - tanh((r - pt->radius) / pt->edge));
}

static const igr_ref2_patch *inflow_patch_for_ghost(const igr_ref2_solver *s, int i, int j, int k, double *weight)
{
    int idx[3] = { i, j, k }, n[3] = { s->nx, s->ny, s->nz };
    for (int a = 0; a < 3; ++a) {
        int face = -1;
        if (idx[a] < 0) face = 2 * a; else if (idx[a] >= n[a]) face = 2 * a + 1;
        if (face < 0 || s->face[face] != IGR_REF_BC_INFLOW) continue;
        int t0 = (a == 0) ? idx[1] : idx[0];
        int t1 = (a == 2) ? idx[1] : idx[2];
        const igr_ref2_patch *best = NULL;
        *weight = 0.0;
        for (int m = 0; m < s->n_patches[face]; ++m) {
            double w = patch_weight(&s->patches[face][m], t0, t1);
            if (w > *weight) { *weight = w; best = &s->patches[face][m]; }
        }
        if (best) return best;
    }
    *weight = 0.0;
    return NULL;
}

/* Step 1: ghosts of the seven fields, then cell-centred mixture density and primitives everywhere. */
int igr_ref2_fill_ghosts(igr_ref2_solver *s)
{
    if (!s) return -1;
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    #pragma omp parallel for
    for (int k = -NG; k < nz + NG; ++k)
        for (int j = -NG; j < ny + NG; ++j)
            for (int i = -NG; i < nx + NG; ++i) {
                if (i >= 0 && i < nx && j >= 0 && j < ny && k >= 0 && k < nz) continue;
                long id = IDX(s, i, j, k);
                double wgt;
                const igr_ref2_patch *pt = inflow_patch_for_ghost(s, i, j, k, &wgt);
                long src = IDX(s, map_index(i, nx, s->face[0]), map_index(j, ny, s->face[2]),
                               map_index(k, nz, s->face[4]));
                if (pt) {
                    double rho = pt->a1rho1 + pt->a2rho2;
                    double ke = 0.5 * rho * (pt->u * pt->u + pt->v * pt->v + pt->w * pt->w);
                    double v[NF] = { pt->a1rho1, pt->a2rho2, rho * pt->u, rho * pt->v, rho * pt->w,
                                     pt->p * big_gamma(s, pt->a1) + ke, pt->a1 };
                    for (int c = 0; c < NF; ++c)
                        s->q[c][id] = wgt >= 1.0 ? v[c] : s->q[c][src] + wgt * (v[c] - s->q[c][src]);
                } else {
                    for (int c = 0; c < NF; ++c) s->q[c][id] = s->q[c][src];
                }
            }
    #pragma omp parallel for
    for (long id = 0; id < s->np; ++id) {
        double rho = s->q[0][id] + s->q[1][id];
        double mx = s->q[2][id], my = s->q[3][id], mz = s->q[4][id], E = s->q[5][id];
        double G = big_gamma(s, s->q[6][id]);
        s->rho[id] = rho;
        s->u[0][id] = mx / rho; s->u[1][id] = my / rho; s->u[2][id] = mz / rho;
        s->p[id] = (1.0 / G) * (E - 0.5 * (mx * mx + my * my + mz * mz) / rho);
        s->c[id] = sqrt((1.0 + 1.0 / G) * s->p[id] / rho);
    }
    return 0;
}

static void fill_sigma_ghosts(igr_ref2_solver *s)
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    #pragma omp parallel for
    for (int k = -NG; k < nz + NG; ++k)
        for (int j = -NG; j < ny + NG; ++j)
            for (int i = -NG; i < nx + NG; ++i) {
                if (i >= 0 && i < nx && j >= 0 && j < ny && k >= 0 && k < nz) continue;
                long src = IDX(s, map_index(i, nx, s->face[0]), map_index(j, ny, s->face[2]),
                               map_index(k, nz, s->face[4]));
                s->sig[IDX(s, i, j, k)] = s->sig[src];
            }
}

/* Steps 2 and 3: eq. (9) with the mixture density and velocity (identical to igr_ref.c). */
int igr_ref2_source(igr_ref2_solver *s)
{
    if (!s) return -1;
    const long st[3] = { s->sx, s->sy, s->sz };
    const double inv2dx = 1.0 / (2.0 * s->dx);
    #pragma omp parallel for
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) {
                long id = IDX(s, i, j, k);
                double G[3][3];
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        G[a][b] = (s->u[a][id + st[b]] - s->u[a][id - st[b]]) * inv2dx;
                double tr_sq = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) tr_sq += G[a][b] * G[b][a];
                double tr = G[0][0] + G[1][1] + G[2][2];
                s->b[id] = s->alpha * (tr_sq + tr * tr);
            }
    return 0;
}

int igr_ref2_solve_sigma(igr_ref2_solver *s)
{
    if (!s) return -1;
    const long st[3] = { s->sx, s->sy, s->sz };
    const double k2 = s->alpha / (s->dx * s->dx);
    for (int it = 0; it < s->n_jacobi; ++it) {
        fill_sigma_ghosts(s);
        #pragma omp parallel for
        for (int k = 0; k < s->nz; ++k)
            for (int j = 0; j < s->ny; ++j)
                for (int i = 0; i < s->nx; ++i) {
                    long id = IDX(s, i, j, k);
                    double num = 0.0, den = 0.0;
                    for (int a = 0; a < 3; ++a)
                        for (int sgn = -1; sgn <= 1; sgn += 2) {
                            long nb = id + sgn * st[a];
                            double w = 2.0 / (s->rho[id] + s->rho[nb]);
                            num += w * s->sig[nb];
                            den += w;
                        }
                    s->sig2[id] = (s->b[id] + k2 * num) / (1.0 / s->rho[id] + k2 * den);
                }
        double *t = s->sig; s->sig = s->sig2; s->sig2 = t;
    }
    fill_sigma_ghosts(s);
    return 0;
}

/* Physical flux of one side along d from the reconstructed conservative values U[0..6] and Sigma; also
 * returns the side's normal velocity. */
static double physical_flux(const igr_ref2_solver *s, int d, const double *U, double sig, double *F)
{
    double rho = U[0] + U[1], E = U[5];
    double ud = U[2 + d] / rho;
    double p = (1.0 / big_gamma(s, U[6])) * (E - 0.5 * (U[2] * U[2] + U[3] * U[3] + U[4] * U[4]) / rho);
    F[0] = (U[0] / rho) * U[2 + d];
    F[1] = (U[1] / rho) * U[2 + d];
    for (int a = 0; a < 3; ++a) F[2 + a] = U[2 + a] * ud + ((a == d) ? (p + sig) : 0.0);
    F[5] = (E + p + sig) * ud;
    F[6] = U[6] * ud;
    return ud;
}

int igr_ref2_rhs(igr_ref2_solver *s)
{
    if (!s) return -1;
    const int n[3] = { s->nx, s->ny, s->nz };
    const long st[3] = { s->sx, s->sy, s->sz };
    for (int c = 0; c < NF; ++c) memset(s->r[c], 0, sizeof(double) * s->np);
    for (int d = 0; d < 3; ++d) {
        int lo[3] = { 0, 0, 0 }, hi[3] = { n[0], n[1], n[2] };
        lo[d] = -1;
        #pragma omp parallel for
        for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i) {
                    long id = IDX(s, i, j, k);          /* left cell of the face */
                    double UL[NF], UR[NF], sL, sR, f6[6], FL[NF], FR[NF];
                    for (int c = 0; c < NF; ++c) {
                        for (int t = -2; t <= 3; ++t) f6[t + 2] = s->q[c][id + t * st[d]];
                        igr_ref_reconstruct(s->order, f6, &UL[c], &UR[c]);
                    }
                    for (int t = -2; t <= 3; ++t) f6[t + 2] = s->sig[id + t * st[d]];
                    igr_ref_reconstruct(s->order, f6, &sL, &sR);
                    long ir = id + st[d];
                    double lamL = fabs(s->u[d][id]) + s->c[id];
                    double lamR = fabs(s->u[d][ir]) + s->c[ir];
                    double lambda = lamL > lamR ? lamL : lamR;
                    double udL = physical_flux(s, d, UL, sL, FL);
                    double udR = physical_flux(s, d, UR, sR, FR);
                    for (int c = 0; c < NF; ++c)
                        s->flux[c][id] = 0.5 * (FL[c] + FR[c]) - 0.5 * lambda * (UR[c] - UL[c]);
                    s->uhat[id] = 0.5 * (udL + udR);
                }
        #pragma omp parallel for
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    long id = IDX(s, i, j, k);
                    for (int c = 0; c < NF; ++c)
                        s->r[c][id] -= (s->flux[c][id] - s->flux[c][id - st[d]]) / s->dx;
                    s->r[6][id] += s->q[6][id] * (s->uhat[id] - s->uhat[id - st[d]]) / s->dx;
                }
    }
    return 0;
}

int igr_ref2_eval_rhs(igr_ref2_solver *s)
{
    if (!s) return -1;
    igr_ref2_fill_ghosts(s);
    igr_ref2_source(s);
    igr_ref2_solve_sigma(s);
    igr_ref2_rhs(s);
    return 0;
}

int igr_ref2_stage(igr_ref2_solver *s, int stage, double dt)
{
    if (!s || stage < 1 || stage > 3) return -1;
    if (stage == 1)
        for (int c = 0; c < NF; ++c) memcpy(s->qn[c], s->q[c], sizeof(double) * s->np);
    igr_ref2_eval_rhs(s);
    const double b = stage == 1 ? 1.0 : (stage == 2 ? 0.25 : 2.0 / 3.0);
    #pragma omp parallel for
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j) {
            long id = IDX(s, 0, j, k);
            for (int c = 0; c < NF; ++c)
                igr_ref_rk_combine(1.0 - b, s->qn[c] + id, b, s->q[c] + id, dt, s->r[c] + id, s->q[c] + id, s->nx);
        }
    return 0;
}

int igr_ref2_step(igr_ref2_solver *s, double dt)
{
    if (!s) return -1;
    for (int stage = 1; stage <= 3; ++stage) igr_ref2_stage(s, stage, dt);
    return 0;
}

int igr_ref2_max_wavespeed(const igr_ref2_solver *s, double *out)
{
    if (!s || !out) return -1;
    double best = 0.0;
    #pragma omp parallel for reduction(max : best)
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) {
                long id = IDX(s, i, j, k);
                double rho = s->q[0][id] + s->q[1][id];
                double mx = s->q[2][id], my = s->q[3][id], mz = s->q[4][id];
                double G = big_gamma(s, s->q[6][id]);
                double p = (1.0 / G) * (s->q[5][id] - 0.5 * (mx * mx + my * my + mz * mz) / rho);
                double um = fmax(fabs(mx / rho), fmax(fabs(my / rho), fabs(mz / rho)));
                double v = um + sqrt((1.0 + 1.0 / G) * p / rho);
                if (v > best) best = v;
            }
    *out = best;
    return 0;
}
