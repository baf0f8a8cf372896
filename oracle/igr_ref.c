/* igr_ref.c -- fp64 CPU ORACLE (test infrastructure, not the product).  See igr_ref.h.
 *
 * Every function restates one passage of PAPER.md (arXiv 2505.07392) as read in
 * SURVEY.md section 8(c) / DESIGN.md "Readings".  No blocking, fusion or reordering:
 * one loop nest per step of the algorithm, in the paper's order.
 * OpenMP is used on outer cell loops only; results do not depend on it
 * (no reductions except max and the wavespeed, which are order-independent).
 */
#include "igr_ref.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NG IGR_REF_NG

struct igr_ref_solver {
    int nx, ny, nz;          /* interior cells                                         */
    long sx, sy, sz, np;     /* padded strides (sx = 1) and padded size                */
    double dx, gamma, alpha;
    int order, n_jacobi, storage;
    int face[6];
    int n_patches[6];
    igr_ref_patch *patches[6];
    double *q[5];            /* current stage state (padded)                           */
    double *qn[5];           /* state at the start of the step (padded, interior used) */
    double *r[5];            /* RHS                                                    */
    double *u[3], *p, *c;    /* cell-centred primitives incl. ghosts                   */
    double *sig, *sig2, *b;  /* Sigma, Sigma ping-pong, source                         */
    double *flux[5];         /* numerical flux of one axis, stored at the left cell    */
    double mu, zeta;         /* shear and bulk viscosity (0: inviscid Euler)           */
    double *G[9];            /* cell-centred velocity gradient G[3a+b] = du_a/dx_b     */
};

static long IDX(const igr_ref_solver *s, int i, int j, int k)
{   /* (i,j,k) interior-relative, may be in [-NG, n+NG) */
    return (long)(i + NG) + s->sy * (long)(j + NG) + s->sz * (long)(k + NG);
}

/* ---------------------------------------------------------------- storage rounding */
/* Round to nearest even onto a binary format with `pbits` significand bits (incl. the
 * hidden one) and minimum normal exponent emin; values beyond `maxv` become +-inf.
 * SURVEY 8(c) C7.  rint() rounds to nearest even in the default rounding mode. */
static double round_to_format(double x, int pbits, int emin, double maxv)
{
    if (x == 0.0 || isnan(x) || isinf(x)) return x;
    int e;
    (void)frexp(x, &e);            /* |x| = f * 2^e, f in [0.5,1)  => exponent e-1 */
    int ex = e - 1;
    if (ex < emin) ex = emin;      /* subnormal range: fixed quantum               */
    double quantum = ldexp(1.0, ex - (pbits - 1));
    double y = rint(x / quantum) * quantum;
    if (fabs(y) > maxv) y = (x > 0) ? INFINITY : -INFINITY;
    return y;
}

double igr_ref_round_storage(double x, int mode)
{
    switch (mode) {
    case IGR_REF_STORE_F32:  return (double)(float)x;
    case IGR_REF_STORE_F16:  return round_to_format(x, 11, -14, 65504.0);
    case IGR_REF_STORE_BF16: return round_to_format(x, 8, -126, 3.3895313892515355e38);
    default:                 return x;
    }
}

static void round_interior(const igr_ref_solver *s, double *f)
{
    if (s->storage == IGR_REF_STORE_F64) return;
    #pragma omp parallel for
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) {
                long id = IDX(s, i, j, k);
                f[id] = igr_ref_round_storage(f[id], s->storage);
            }
}

/* ---------------------------------------------------------------- create / destroy */
static double *alloc_field(long n)
{
    double *p = (double *)calloc((size_t)n, sizeof(double));
    return p;
}

int igr_ref_create(int nx, int ny, int nz, double dx, double gamma, double alpha,
                   int order, int n_jacobi, const igr_ref_bc *bc, igr_ref_solver **out)
{
    if (!out || !bc || nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(gamma > 1) ||
        alpha < 0 || n_jacobi < 0) return -1;
    if (order != 5 && order != 3) return -1;
    for (int a = 0; a < 3; ++a) {   /* periodic must be on both faces of an axis */
        int lo = bc->face[2 * a], hi = bc->face[2 * a + 1];
        if ((lo == IGR_REF_BC_PERIODIC) != (hi == IGR_REF_BC_PERIODIC)) return -2;
        if (lo < 0 || lo > 3 || hi < 0 || hi > 3) return -2;
    }
    igr_ref_solver *s = (igr_ref_solver *)calloc(1, sizeof(*s));
    if (!s) return -3;
    s->nx = nx; s->ny = ny; s->nz = nz;
    s->sx = 1; s->sy = nx + 2 * NG; s->sz = s->sy * (ny + 2 * NG);
    s->np = s->sz * (nz + 2 * NG);
    s->dx = dx; s->gamma = gamma; s->alpha = alpha;
    s->order = order; s->n_jacobi = n_jacobi; s->storage = IGR_REF_STORE_F64;
    for (int f = 0; f < 6; ++f) {
        s->face[f] = bc->face[f];
        s->n_patches[f] = (bc->face[f] == IGR_REF_BC_INFLOW) ? bc->n_patches[f] : 0;
        if (s->n_patches[f] > 0) {
            s->patches[f] = (igr_ref_patch *)malloc(sizeof(igr_ref_patch) * s->n_patches[f]);
            memcpy(s->patches[f], bc->patches[f], sizeof(igr_ref_patch) * s->n_patches[f]);
        }
    }
    for (int c = 0; c < 5; ++c) {
        s->q[c] = alloc_field(s->np); s->qn[c] = alloc_field(s->np); s->r[c] = alloc_field(s->np);
    }
    for (int a = 0; a < 3; ++a) s->u[a] = alloc_field(s->np);
    s->p = alloc_field(s->np); s->c = alloc_field(s->np);
    s->sig = alloc_field(s->np); s->sig2 = alloc_field(s->np); s->b = alloc_field(s->np);
    for (int c = 0; c < 5; ++c) s->flux[c] = alloc_field(s->np);
    for (int c = 0; c < 9; ++c) s->G[c] = NULL;
    *out = s;
    return 0;
}

void igr_ref_destroy(igr_ref_solver *s)
{
    if (!s) return;
    for (int c = 0; c < 5; ++c) { free(s->q[c]); free(s->qn[c]); free(s->r[c]); free(s->flux[c]); }
    for (int a = 0; a < 3; ++a) free(s->u[a]);
    free(s->p); free(s->c); free(s->sig); free(s->sig2); free(s->b);
    for (int c = 0; c < 9; ++c) free(s->G[c]);
    for (int f = 0; f < 6; ++f) free(s->patches[f]);
    free(s);
}

/* NEXT-1: Newtonian viscous stress, eqs. (2), (3), (5). */
int igr_ref_set_viscosity(igr_ref_solver *s, double mu, double zeta)
{
    if (!s || mu < 0 || zeta < 0) return -1;
    s->mu = mu; s->zeta = zeta;
    if ((mu > 0 || zeta > 0) && !s->G[0])
        for (int c = 0; c < 9; ++c) s->G[c] = alloc_field(s->np);
    return 0;
}

int igr_ref_set_storage(igr_ref_solver *s, int mode)
{
    if (!s || mode < 0 || mode > 3) return -1;
    s->storage = mode;
    return 0;
}

/* ---------------------------------------------------------------- interior copies  */
static void put_interior(const igr_ref_solver *s, double *dst, const double *src)
{
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i)
                dst[IDX(s, i, j, k)] = src[((long)k * s->ny + j) * s->nx + i];
}

static void take_interior(const igr_ref_solver *s, const double *src, double *dst)
{
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i)
                dst[((long)k * s->ny + j) * s->nx + i] = src[IDX(s, i, j, k)];
}

int igr_ref_set_state(igr_ref_solver *s, const double *q)
{
    if (!s || !q) return -1;
    long n = (long)s->nx * s->ny * s->nz;
    for (int c = 0; c < 5; ++c) {
        put_interior(s, s->q[c], q + c * n);
        round_interior(s, s->q[c]);
    }
    memset(s->sig, 0, sizeof(double) * s->np);   /* configs: "Sigma = 0 at t = 0" */
    memset(s->sig2, 0, sizeof(double) * s->np);
    return 0;
}

int igr_ref_get_state(const igr_ref_solver *s, double *q)
{
    if (!s || !q) return -1;
    long n = (long)s->nx * s->ny * s->nz;
    for (int c = 0; c < 5; ++c) take_interior(s, s->q[c], q + c * n);
    return 0;
}

int igr_ref_set_sigma(igr_ref_solver *s, const double *sig)
{
    if (!s || !sig) return -1;
    put_interior(s, s->sig, sig);
    round_interior(s, s->sig);
    return 0;
}

int igr_ref_get_sigma(const igr_ref_solver *s, double *sig)
{
    if (!s || !sig) return -1;
    take_interior(s, s->sig, sig);
    return 0;
}

int igr_ref_get_source(const igr_ref_solver *s, double *b)
{
    if (!s || !b) return -1;
    take_interior(s, s->b, b);
    return 0;
}

int igr_ref_set_source(igr_ref_solver *s, const double *b)
{   /* test hook: drive the Jacobi sweeps with a given right-hand side */
    if (!s || !b) return -1;
    put_interior(s, s->b, b);
    return 0;
}

int igr_ref_get_rhs(const igr_ref_solver *s, double *r)
{
    if (!s || !r) return -1;
    long n = (long)s->nx * s->ny * s->nz;
    for (int c = 0; c < 5; ++c) take_interior(s, s->r[c], r + c * n);
    return 0;
}

int igr_ref_get_padded(const igr_ref_solver *s, int c, double *out)
{
    if (!s || !out || c < 0 || c > 5) return -1;
    memcpy(out, c < 5 ? s->q[c] : s->sig, sizeof(double) * s->np);
    return 0;
}

int igr_ref_set_padded(igr_ref_solver *s, int c, const double *in)
{
    if (!s || !in || c < 0 || c > 5) return -1;
    memcpy(c < 5 ? s->q[c] : s->sig, in, sizeof(double) * s->np);
    return 0;
}

/* ---------------------------------------------------------------- boundary conditions
 * The paper gives no boundary conditions; BASELINE.json names periodic, extrapolation
 * outflow and fixed-state inflow patches.  SURVEY 8(c) "BC as an index map":
 *   periodic      -> wrap modulo n
 *   extrapolation -> clamp to the nearest interior index (zeroth order)
 *   inflow        -> fixed patch state where the ghost cell's transverse centre lies in
 *                    a patch circle (optionally blended over a tanh edge), clamp elsewhere.
 * Sigma: wrap on periodic faces, clamp on every other face (homogeneous Neumann). */
static int map_index(int i, int n, int face_lo)
{
    if (i >= 0 && i < n) return i;
    if (face_lo == IGR_REF_BC_PERIODIC) { int m = i % n; return m < 0 ? m + n : m; }
    return i < 0 ? 0 : n - 1;
}

/* Weight in [0,1] of patch `pt` at the transverse cell centre (t0+1/2, t1+1/2):
 *   edge == 0: 1 inside the circle r <= radius, 0 outside (sharp mask);
 *   edge  > 0: (1 - tanh((r - radius)/edge))/2, cut to exactly 0 for r >= radius + 4 edge
 * (reading A8b: a grid-sharp patch edge is not survivable by the purely linear scheme). */
static double patch_weight(const igr_ref_patch *pt, int t0, int t1)
{
    double d0 = (t0 + 0.5) - pt->c0, d1 = (t1 + 0.5) - pt->c1;
    double r2 = d0 * d0 + d1 * d1;
    if (pt->edge <= 0.0) return (r2 <= pt->radius * pt->radius) ? 1.0 : 0.0;
    double r = sqrt(r2);
    if (r >= pt->radius + 4.0 * pt->edge) return 0.0;
    return 0.5 * (1.0 - tanh((r - pt->radius) / pt->edge));
}

/* the patch with the largest weight at this transverse position (first wins ties) */
static const igr_ref_patch *find_patch(const igr_ref_solver *s, int face, int t0, int t1,
                                       double *weight)
{
    const igr_ref_patch *best = NULL;
    *weight = 0.0;
    for (int n = 0; n < s->n_patches[face]; ++n) {
        double w = patch_weight(&s->patches[face][n], t0, t1);
        if (w > *weight) { *weight = w; best = &s->patches[face][n]; }
    }
    return best;
}

/* Domain decomposition (reading A20): a ghost cell that lies beyond an EXTERNAL face along any of its
 * out-of-range axes belongs to the neighbouring sub-domain (or is an edge/corner cell no stencil reads):
 * it is never written here. */
static int ghost_is_external(const igr_ref_solver *s, int i, int j, int k)
{
    int idx[3] = { i, j, k }, n[3] = { s->nx, s->ny, s->nz };
    for (int a = 0; a < 3; ++a) {
        if (idx[a] < 0 && s->face[2 * a] == IGR_REF_BC_EXTERNAL) return 1;
        if (idx[a] >= n[a] && s->face[2 * a + 1] == IGR_REF_BC_EXTERNAL) return 1;
    }
    return 0;
}

static const igr_ref_patch *inflow_patch_for_ghost(const igr_ref_solver *s, int i, int j, int k,
                                                   double *weight)
{
    int idx[3] = { i, j, k }, n[3] = { s->nx, s->ny, s->nz };
    for (int a = 0; a < 3; ++a) {
        int face = -1;
        if (idx[a] < 0) face = 2 * a; else if (idx[a] >= n[a]) face = 2 * a + 1;
        if (face < 0 || s->face[face] != IGR_REF_BC_INFLOW) continue;
        int t0 = (a == 0) ? idx[1] : idx[0];          /* transverse axes in x<y<z order */
        int t1 = (a == 2) ? idx[1] : idx[2];
        const igr_ref_patch *pt = find_patch(s, face, t0, t1, weight);
        if (pt) return pt;
    }
    *weight = 0.0;
    return NULL;
}

/* Step 1 of SURVEY 8(c): fill ghosts of q, then cell-centred primitives everywhere.
 * u = m/rho, p = (gamma-1)(E - |m|^2/(2 rho))  (eq. 4), c = sqrt(gamma p/rho). */
int igr_ref_fill_ghosts(igr_ref_solver *s)
{
    if (!s) return -1;
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    #pragma omp parallel for
    for (int k = -NG; k < nz + NG; ++k)
        for (int j = -NG; j < ny + NG; ++j)
            for (int i = -NG; i < nx + NG; ++i) {
                if (i >= 0 && i < nx && j >= 0 && j < ny && k >= 0 && k < nz) continue;
                if (ghost_is_external(s, i, j, k)) continue;
                long id = IDX(s, i, j, k);
                double wgt;
                const igr_ref_patch *pt = inflow_patch_for_ghost(s, i, j, k, &wgt);
                long src = IDX(s, map_index(i, nx, s->face[0]), map_index(j, ny, s->face[2]),
                               map_index(k, nz, s->face[4]));
                if (pt) {     /* ghost = interior + w * (fixed - interior): w = 1 gives the fixed
                               * state exactly, fixed == interior gives it back exactly */
                    double ke = 0.5 * pt->rho * (pt->u * pt->u + pt->v * pt->v + pt->w * pt->w);
                    double v[5] = { pt->rho, pt->rho * pt->u, pt->rho * pt->v, pt->rho * pt->w,
                                    pt->p / (s->gamma - 1.0) + ke };
                    for (int c = 0; c < 5; ++c)
                        s->q[c][id] = igr_ref_round_storage(
                            wgt >= 1.0 ? v[c] : s->q[c][src] + wgt * (v[c] - s->q[c][src]),
                            s->storage);
                } else {
                    for (int c = 0; c < 5; ++c) s->q[c][id] = s->q[c][src];
                }
            }
    #pragma omp parallel for
    for (long id = 0; id < s->np; ++id) {
        double rho = s->q[0][id], mx = s->q[1][id], my = s->q[2][id], mz = s->q[3][id], E = s->q[4][id];
        s->u[0][id] = mx / rho; s->u[1][id] = my / rho; s->u[2][id] = mz / rho;
        s->p[id] = (s->gamma - 1.0) * (E - 0.5 * (mx * mx + my * my + mz * mz) / rho);
        s->c[id] = sqrt(s->gamma * s->p[id] / rho);
    }
    return 0;
}

int igr_ref_fill_sigma_ghosts(igr_ref_solver *s)
{
    if (!s) return -1;
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    #pragma omp parallel for
    for (int k = -NG; k < nz + NG; ++k)
        for (int j = -NG; j < ny + NG; ++j)
            for (int i = -NG; i < nx + NG; ++i) {
                if (i >= 0 && i < nx && j >= 0 && j < ny && k >= 0 && k < nz) continue;
                if (ghost_is_external(s, i, j, k)) continue;
                long src = IDX(s, map_index(i, nx, s->face[0]), map_index(j, ny, s->face[2]),
                               map_index(k, nz, s->face[4]));
                s->sig[IDX(s, i, j, k)] = s->sig[src];
            }
    return 0;
}

/* ---------------------------------------------------------------- step 2: source
 * b = alpha * ( tr((grad u)^2) + (tr grad u)^2 ), left side of eq. (9) as printed
 * (footnote L252), with second-order central differences of the
 * cell-centred velocity (L132; Alg. 1):  G_ab = d u_a / d x_b. */
int igr_ref_source(igr_ref_solver *s)
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
                double tr_sq = 0.0;                      /* tr(G G) = sum_ab G_ab G_ba */
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) tr_sq += G[a][b] * G[b][a];
                double tr = G[0][0] + G[1][1] + G[2][2];
                s->b[id] = s->alpha * (tr_sq + tr * tr);
            }
    return 0;
}

/* ---------------------------------------------------------------- step 3: Jacobi
 * Sigma/rho - alpha div( grad(Sigma)/rho ) = b   (eq. 9, reading A1), "standard 6-point
 * stencil" (L138) with face density = arithmetic mean (reading A2):
 *   Sigma_i <- ( b_i + (alpha/dx^2) sum_n w_in Sigma_n ) / ( 1/rho_i + (alpha/dx^2) sum_n w_in ),
 *   w_in = 2 / (rho_i + rho_n),  n over the six face neighbours.
 * One call = refresh the ghosts of the current iterate, then one sweep (L130, L138). */
int igr_ref_jacobi_sweep(igr_ref_solver *s)
{
    if (!s) return -1;
    igr_ref_fill_sigma_ghosts(s);
    const long st[3] = { s->sx, s->sy, s->sz };
    const double k2 = s->alpha / (s->dx * s->dx);
    const double *rho = s->q[0];
    #pragma omp parallel for
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) {
                long id = IDX(s, i, j, k);
                double num = 0.0, den = 0.0;
                for (int a = 0; a < 3; ++a)
                    for (int sgn = -1; sgn <= 1; sgn += 2) {
                        long nb = id + sgn * st[a];
                        double w = 2.0 / (rho[id] + rho[nb]);
                        num += w * s->sig[nb];
                        den += w;
                    }
                s->sig2[id] = (s->b[id] + k2 * num) / (1.0 / rho[id] + k2 * den);
            }
    double *t = s->sig; s->sig = s->sig2; s->sig2 = t;
    return 0;
}

int igr_ref_solve_sigma(igr_ref_solver *s)
{
    if (!s) return -1;
    for (int it = 0; it < s->n_jacobi; ++it) igr_ref_jacobi_sweep(s);
    round_interior(s, s->sig);                   /* storage emulation (C7) */
    igr_ref_fill_sigma_ghosts(s);
    return 0;
}

/* ---------------------------------------------------------------- step 4: reconstruction
 * Fifth-order accurate linear finite-volume reconstruction of cell averages at the face
 * between cells 0 and 1 from the stencil cells -2..3 (Alg. 1,
 * L183-L196).  f6[q+2] holds cell q.  Upwind-biased optimal linear weights:
 *   f_L = ( 2 f_-2 - 13 f_-1 + 47 f_0 + 27 f_1 -  3 f_2) / 60
 *   f_R = (-3 f_-1 + 27 f_0  + 47 f_1 - 13 f_2 +  2 f_3) / 60
 * order 3 (optional):  f_L = (-f_-1 + 5 f_0 + 2 f_1)/6,  f_R = (2 f_0 + 5 f_1 - f_2)/6. */
void igr_ref_reconstruct(int order, const double *f6, double *fL, double *fR)
{
    const double *f = f6 + 2;       /* f[q], q = -2..3 */
    if (order == 5) {
        *fL = ( 2.0 * f[-2] - 13.0 * f[-1] + 47.0 * f[0] + 27.0 * f[1] -  3.0 * f[2]) / 60.0;
        *fR = (-3.0 * f[-1] + 27.0 * f[0]  + 47.0 * f[1] - 13.0 * f[2] +  2.0 * f[3]) / 60.0;
    } else {
        *fL = (-f[-1] + 5.0 * f[0] + 2.0 * f[1]) / 6.0;
        *fR = ( 2.0 * f[0] + 5.0 * f[1] - f[2]) / 6.0;
    }
}

/* ---------------------------------------------------------------- steps 5-6: LF flux
 * Face primitives from the RECONSTRUCTED conservative values (Alg. 1):
 *   u = m/rho,  p = (gamma-1)(E - |m|^2/(2 rho)).
 * Physical flux along d with the entropic pressure added to p (eqs. 6-8):
 *   F = ( m_d, m_x u_d + (p+Sigma) d_xd, m_y u_d + (p+Sigma) d_yd, m_z u_d + (p+Sigma) d_zd,
 *         (E + p + Sigma) u_d ).
 * Lax-Friedrichs (L132, Alg. 1):  F^ = (F_L + F_R)/2 - lambda (U_R - U_L)/2. */
static void physical_flux(int d, double gamma, const double *U, double sig, double *F)
{
    double rho = U[0], E = U[4];
    double u[3] = { U[1] / rho, U[2] / rho, U[3] / rho };
    double p = (gamma - 1.0) * (E - 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / rho);
    double ud = u[d];
    F[0] = U[1 + d];
    for (int a = 0; a < 3; ++a) F[1 + a] = U[1 + a] * ud + ((a == d) ? (p + sig) : 0.0);
    F[4] = (E + p + sig) * ud;
}

void igr_ref_lf_flux(int d, double gamma, const double *UL, const double *UR,
                     double sigL, double sigR, double lambda, double *F)
{
    double FL[5], FR[5];
    physical_flux(d, gamma, UL, sigL, FL);
    physical_flux(d, gamma, UR, sigR, FR);
    for (int c = 0; c < 5; ++c)
        F[c] = 0.5 * (FL[c] + FR[c]) - 0.5 * lambda * (UR[c] - UL[c]);
}

/* ---------------------------------------------------------------- viscous fluxes (NEXT-1)
 * Second-order velocity gradients (L132), the same ones the Sigma source uses (L232), at the
 * cell centres: G_ab = (u_a[i+e_b] - u_a[i-e_b]) / (2 dx) on the interior; ghosts of this derived
 * field by the BC index map (wrap / clamp; reading A19).  They are reconstructed at the face with
 * the reconstruction coefficients of the state (Alg. 1: vflux_L/R += coeff_L/R(q) du/dn),
 * the face velocity comes from the reconstructed conservative state (L187-L189), and the two
 * sides are averaged (reading A19: the paper only names `viscous(vflux_L, vflux_R, u_L, u_R)`):
 *   tau_ab = mu (G_ab + G_ba) + (zeta - 2 mu / 3) delta_ab tr G                    (eq. 5)
 *   F_visc along d = ( 0, -tau_xd, -tau_yd, -tau_zd, -(u . tau)_d )               (eqs. 2-3)   */
static void velocity_gradients(igr_ref_solver *s)
{
    const long st[3] = { s->sx, s->sy, s->sz };
    const double inv2dx = 1.0 / (2.0 * s->dx);
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    #pragma omp parallel for
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                long id = IDX(s, i, j, k);
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b)
                        s->G[3 * a + b][id] = (s->u[a][id + st[b]] - s->u[a][id - st[b]]) * inv2dx;
            }
    #pragma omp parallel for
    for (int k = -NG; k < nz + NG; ++k)
        for (int j = -NG; j < ny + NG; ++j)
            for (int i = -NG; i < nx + NG; ++i) {
                if (i >= 0 && i < nx && j >= 0 && j < ny && k >= 0 && k < nz) continue;
                if (ghost_is_external(s, i, j, k)) continue;
                long src = IDX(s, map_index(i, nx, s->face[0]), map_index(j, ny, s->face[2]),
                               map_index(k, nz, s->face[4]));
                for (int c = 0; c < 9; ++c) s->G[c][IDX(s, i, j, k)] = s->G[c][src];
            }
}

/* viscous flux along d from the face values of the gradient tensor and the velocity */
void igr_ref_viscous_flux(int d, double mu, double zeta, const double *G9, const double *u3, double *F)
{
    double tr = G9[0] + G9[4] + G9[8];
    double tau[3];                                   /* tau_ad, a = x, y, z */
    for (int a = 0; a < 3; ++a)
        tau[a] = mu * (G9[3 * a + d] + G9[3 * d + a]) + ((a == d) ? (zeta - 2.0 * mu / 3.0) * tr : 0.0);
    F[0] = 0.0;
    for (int a = 0; a < 3; ++a) F[1 + a] = -tau[a];
    F[4] = -(u3[0] * tau[0] + u3[1] * tau[1] + u3[2] * tau[2]);
}

/* ---------------------------------------------------------------- steps 4-7: RHS
 * For each axis d (dimensional splitting, Alg. 1) and each face i+1/2 bounding an
 * interior cell: reconstruct the six fields (q and Sigma, Alg. 1 L183-L196, L205/L224),
 * LF flux with lambda = max(|u_d|+c) over the two adjacent CELL-CENTRED states (reading
 * A5), then r_i = - sum_d (F^_{i+1/2,d} - F^_{i-1/2,d}) / dx. */
int igr_ref_rhs(igr_ref_solver *s)
{
    if (!s) return -1;
    const int n[3] = { s->nx, s->ny, s->nz };
    const long st[3] = { s->sx, s->sy, s->sz };
    for (int c = 0; c < 5; ++c) memset(s->r[c], 0, sizeof(double) * s->np);
    const int viscous = (s->mu > 0 || s->zeta > 0);
    if (viscous) velocity_gradients(s);
    for (int d = 0; d < 3; ++d) {
        /* faces: left cell index along d runs -1..n_d-1, other axes over the interior */
        int lo[3] = { 0, 0, 0 }, hi[3] = { n[0], n[1], n[2] };
        lo[d] = -1;
        #pragma omp parallel for
        for (int k = lo[2]; k < hi[2]; ++k)
            for (int j = lo[1]; j < hi[1]; ++j)
                for (int i = lo[0]; i < hi[0]; ++i) {
                    long id = IDX(s, i, j, k);          /* left cell of the face */
                    double UL[5], UR[5], sL, sR, f6[6];
                    for (int c = 0; c < 5; ++c) {
                        for (int t = -2; t <= 3; ++t) f6[t + 2] = s->q[c][id + t * st[d]];
                        igr_ref_reconstruct(s->order, f6, &UL[c], &UR[c]);
                    }
                    for (int t = -2; t <= 3; ++t) f6[t + 2] = s->sig[id + t * st[d]];
                    igr_ref_reconstruct(s->order, f6, &sL, &sR);
                    long ir = id + st[d];
                    double lamL = fabs(s->u[d][id]) + s->c[id];
                    double lamR = fabs(s->u[d][ir]) + s->c[ir];
                    double lambda = lamL > lamR ? lamL : lamR;
                    double F[5];
                    igr_ref_lf_flux(d, s->gamma, UL, UR, sL, sR, lambda, F);
                    if (viscous) {
                        double GL[9], GR[9], Gf[9], uf[3], Fv[5];
                        for (int c = 0; c < 9; ++c) {
                            for (int t = -2; t <= 3; ++t) f6[t + 2] = s->G[c][id + t * st[d]];
                            igr_ref_reconstruct(s->order, f6, &GL[c], &GR[c]);
                            Gf[c] = 0.5 * (GL[c] + GR[c]);
                        }
                        for (int a = 0; a < 3; ++a) uf[a] = 0.5 * (UL[1 + a] / UL[0] + UR[1 + a] / UR[0]);
                        igr_ref_viscous_flux(d, s->mu, s->zeta, Gf, uf, Fv);
                        for (int c = 0; c < 5; ++c) F[c] += Fv[c];
                    }
                    for (int c = 0; c < 5; ++c) s->flux[c][id] = F[c];
                }
        #pragma omp parallel for
        for (int k = 0; k < n[2]; ++k)
            for (int j = 0; j < n[1]; ++j)
                for (int i = 0; i < n[0]; ++i) {
                    long id = IDX(s, i, j, k);
                    for (int c = 0; c < 5; ++c)
                        s->r[c][id] -= (s->flux[c][id] - s->flux[c][id - st[d]]) / s->dx;
                }
    }
    return 0;
}

int igr_ref_eval_rhs(igr_ref_solver *s)
{
    if (!s) return -1;
    igr_ref_fill_ghosts(s);
    igr_ref_source(s);
    igr_ref_solve_sigma(s);
    igr_ref_rhs(s);
    return 0;
}

/* ---------------------------------------------------------------- time stepping
 * Third-order SSP (TVD) Runge-Kutta of Gottlieb & Shu (ref. 17 L389):
 *   q1 = qn + dt L(qn);  q2 = 3/4 qn + 1/4 (q1 + dt L(q1));  qn+1 = 1/3 qn + 2/3 (q2 + dt L(q2)).
 * Each stage is a*qn + b*(qs + dt r) with a + b = 1; it is evaluated as
 *   qn + b*((qs - qn) + dt r)
 * (same value in exact arithmetic) so that r = 0, qs = qn returns qn bitwise
 * (reading A18: uniform states are preserved exactly). */
void igr_ref_rk_combine(double a, const double *qn, double b, const double *qs,
                        double dt, const double *r, double *out, long n)
{
    (void)a;                                   /* a = 1 - b */
    for (long i = 0; i < n; ++i) out[i] = qn[i] + b * ((qs[i] - qn[i]) + dt * r[i]);
}

static void rk_stage(igr_ref_solver *s, double a, double b, double dt)
{
    #pragma omp parallel for
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j) {
            long id = IDX(s, 0, j, k);
            for (int c = 0; c < 5; ++c)
                igr_ref_rk_combine(a, s->qn[c] + id, b, s->q[c] + id, dt, s->r[c] + id,
                                   s->q[c] + id, s->nx);
        }
    for (int c = 0; c < 5; ++c) round_interior(s, s->q[c]);   /* storage emulation (C7) */
}

/* Sigma is a persistent field: each of the three solves is warm-started from the
 * previous one (L130, L138; reading A4); it is not RK-combined. */
int igr_ref_stage(igr_ref_solver *s, int stage, double dt)
{
    if (!s || stage < 1 || stage > 3) return -1;
    if (stage == 1)
        for (int c = 0; c < 5; ++c) memcpy(s->qn[c], s->q[c], sizeof(double) * s->np);
    igr_ref_eval_rhs(s);
    if (stage == 1) rk_stage(s, 0.0, 1.0, dt);
    else if (stage == 2) rk_stage(s, 0.75, 0.25, dt);
    else rk_stage(s, 1.0 / 3.0, 2.0 / 3.0, dt);
    return 0;
}

int igr_ref_step(igr_ref_solver *s, double dt)
{
    if (!s) return -1;
    for (int stage = 1; stage <= 3; ++stage) igr_ref_stage(s, stage, dt);
    return 0;
}

/* max over interior cells of max(|u|,|v|,|w|) + c  (CFL condition, reading A9) */
int igr_ref_max_wavespeed(const igr_ref_solver *s, double *out)
{
    if (!s || !out) return -1;
    double best = 0.0;
    #pragma omp parallel for reduction(max : best)
    for (int k = 0; k < s->nz; ++k)
        for (int j = 0; j < s->ny; ++j)
            for (int i = 0; i < s->nx; ++i) {
                long id = IDX(s, i, j, k);
                double rho = s->q[0][id], mx = s->q[1][id], my = s->q[2][id], mz = s->q[3][id];
                double p = (s->gamma - 1.0) * (s->q[4][id] - 0.5 * (mx * mx + my * my + mz * mz) / rho);
                double um = fmax(fabs(mx / rho), fmax(fabs(my / rho), fabs(mz / rho)));
                double v = um + sqrt(s->gamma * p / rho);
                if (v > best) best = v;
            }
    *out = best;
    return 0;
}
