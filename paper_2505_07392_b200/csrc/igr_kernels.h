// igr_kernels.h -- host-side launchers of the CUDA kernels of libigr (one per row of the hot path,
// SURVEY.md 8(a)).  `storage` is IGR_STORE_F32 / F16 / BF16 (igr.h); q and Sigma use that element
// type, b and r are always fp32.
#pragma once
#include <cuda.h>
#include "igr_common.cuh"

struct RhsParams {
    float gamma, inv_dx;
    int order;
};

// interior <-> padded copies.  `user` is a DEVICE fp32 array holding planes [k0, k0+nk) of one
// field, layout [nk][ny][nx].
void launch_unpack_field(const Grid &g, int storage, const float *user, void *field, int k0, int nk,
                         cudaStream_t st);
void launch_pack_field(const Grid &g, int storage, const void *field, float *user, int k0, int nk,
                       cudaStream_t st);
void launch_unpack_f32(const Grid &g, const float *user, float *field, int k0, int nk, cudaStream_t st);
void launch_pack_f32(const Grid &g, const float *field, float *user, int k0, int nk, cudaStream_t st);
// padded copy with 3 ghost layers: out [nz+6][ny+6][nx+6] planes [k0,k0+nk) of the padded z range
void launch_pack_padded(const Grid &g, int storage, const void *field, float *user, int k0, int nk,
                        cudaStream_t st);

// a1: ghosts of q (5 fields) / of Sigma
// (nf = 5 fields, or 7 with two fluids; the fixed inflow states hold nf values per transverse cell)
void launch_halo_q(const Grid &g, int storage, StagePtrs q, const BcDesc &bc, int nf, cudaStream_t st);
// two fluids (NEXT-3, reading A21; fp32 storage): mixture density of every cell of the padded array, and the
// mixture wave speed
void launch_rho_total(const Grid &g, const float *r1, const float *r2, float *out, cudaStream_t st);
void launch_wavespeed2(const Grid &g, StagePtrs q, float k1, float k2, WaveResult *wave, cudaStream_t st);
void launch_halo_sigma(const Grid &g, int storage, void *sig, cudaStream_t st);

// a2: b = alpha (tr((grad u)^2) + (tr grad u)^2)
// `tau` (block of 6 fp32 padded fields, stride g.np: the viscous stress of eq. 5, igr_viscous.cuh) is
// also written when not NULL
void launch_source(const Grid &g, int storage, StagePtrs q, float *b, float alpha, float inv2dx,
                   float *tau, float mu, float zeta, cudaStream_t st);
// a2, TMA-staged form (igr_source_tma.cu): b only (the stress fields of the viscous variant stay with launch_source).
// f: the padded fields rho, m_x, m_y, m_z in the storage type (two fluids: rho = the fp32 mixture density).
struct SourceMaps {
    CUtensorMap f[4];
    bool valid;
};
int source_make_maps(const Grid &g, int storage, void *const f[4], SourceMaps *out);
void launch_source_tma(const Grid &g, int storage, const SourceMaps &m, float *b, float alpha, float inv2dx,
                       cudaStream_t st);
// ghosts of nf derived fp32 fields (stride g.np) by the BC index map
void launch_halo_fields(const Grid &g, float *base, int nf, cudaStream_t st);
// NEXT-1, simple form: r[1..4] += -div F_visc (eqs. 2, 3, 5); tau must have its ghosts filled
void launch_viscous_add(const Grid &g, int storage, int order, StagePtrs q, const float *tau,
                        float *const r[5], float inv_dx, cudaStream_t st);

// a3 (simple form): one Jacobi sweep, neighbours of Sigma through the BC index map
void launch_jacobi_sweep(const Grid &g, int storage, const void *rho, const float *b,
                         const void *sig_in, void *sig_out, float k2, cudaStream_t st);

// a4 (simple form): r = -div F^
void launch_rhs_simple(const Grid &g, int storage, StagePtrs q, const void *sig, float *const r[5],
                       RhsParams p, cudaStream_t st);

// a5: q_out = q_n + beta ((q_s - q_n) + dt r); if `wave` != NULL also reduces the wave speed of q_out
void launch_rk_update(const Grid &g, int storage, StagePtrs qn, StagePtrs qs, StagePtrs qout,
                      float *const r[5], float beta, float dt, float gamma, WaveResult *wave,
                      cudaStream_t st);

// a6: wave = max_cells(max_d |u_d| + c), non-finite flag
void launch_wavespeed(const Grid &g, int storage, StagePtrs q, float gamma, WaveResult *wave,
                      cudaStream_t st);

// a3 (blocked form): ns in 1..5 sweeps in ONE pass over HBM (igr_jacobi_blocked.cu); sig_in != sig_out.
// TMA maps of the planes of rho (the three state buffers), Sigma (two buffers) and b: regions inside the
// domain stage their planes with them; NULL maps: every region gathers with cp.async.
struct JacobiMaps {
    CUtensorMap rho[3], sig[2], b;
    bool valid;
};
// rows: box height (32: the blocked kernel and quad regions 22 rows apart; 34: quad regions 24 rows apart)
int jacobi_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state, void *const sig[2],
                     const float *b, JacobiMaps *out, int rows = 32);
// a3 (quad form, igr_jacobi_quad.cu): the same blocked pass for the regions (bx, by), bx0 <= bx < bx0 + nbx,
// by0 <= by < by0 + nby, that need no periodic wrap in x / y; four y-adjacent columns per thread.  nbx = 0: none.
struct JacobiQuadPlan {
    int bx0, by0, nbx, nby, zc;
    int wy, nby_blocked;   // wy: regions 24 rows apart with 34-row boxes (TMA maps of jacobi_make_maps(..., rows = 34));
};                         // nby_blocked: the same y range counted in regions of the blocked kernel's grid (skip test)
JacobiQuadPlan jacobi_quad_plan(const Grid &g, int ns, float k2);
void launch_jacobi_quad(const Grid &g, int storage, int ns, const JacobiQuadPlan &pl, void *sig_out, float k2,
                        const CUtensorMap *rmap, const CUtensorMap *bmap, const CUtensorMap *smap, cudaStream_t st);
// `skip` (may be NULL): regions of that plan are left to launch_jacobi_quad
void launch_jacobi_blocked(const Grid &g, int storage, int ns, const void *rho, const float *b,
                           const void *sig_in, void *sig_out, float k2, const CUtensorMap *rmap,
                           const CUtensorMap *bmap, const CUtensorMap *smap, const JacobiQuadPlan *skip,
                           cudaStream_t st);

// ---- fp64 mode (IGR_STORE_F64, NEXT-4): fp64 storage and arithmetic, one thread per cell, one launch per row and
// per sweep (igr_kernels.cu, namespace f64).  `user` arrays are fp64 or fp32 (user_is_f32).
void launch64_unpack(const Grid &g, const void *user, int user_is_f32, double *field, int k0, int nk, cudaStream_t st);
void launch64_pack(const Grid &g, const double *field, void *user, int user_is_f32, int k0, int nk, cudaStream_t st);
void launch64_halo_q(const Grid &g, StagePtrs q, const Inflow64 &bc, cudaStream_t st);
void launch64_halo_sigma(const Grid &g, double *sig, cudaStream_t st);
void launch64_source(const Grid &g, StagePtrs q, double *b, double alpha, double inv2dx, cudaStream_t st);
void launch64_jacobi_sweep(const Grid &g, const double *rho, const double *b, const double *sin, double *sout, double k2,
                           cudaStream_t st);
void launch64_rhs(const Grid &g, int order, StagePtrs q, const double *sig, double *const r[5], double gamma, double dx,
                  cudaStream_t st);
void launch64_rk_update(const Grid &g, StagePtrs qn, StagePtrs qs, StagePtrs qout, double *const r[5], double beta,
                        double dt, double gamma, WaveResult64 *wave, cudaStream_t st);
void launch64_wavespeed(const Grid &g, StagePtrs q, double gamma, WaveResult64 *wave, cudaStream_t st);
