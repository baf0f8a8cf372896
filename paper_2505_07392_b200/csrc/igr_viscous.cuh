// igr_viscous.cuh -- NEXT-1: Newtonian viscous fluxes, eqs. (2), (3), (5) (
// Alg. 1; reading A19).
//
// The source kernel (row a2) already forms the second-order velocity gradients G_ab = du_a/dx_b at the
// cell centres (L132, L232).  It stores the six components of the symmetric stress
//   tau_ab = mu (G_ab + G_ba) + (zeta - 2 mu / 3) delta_ab tr G                                  (eq. 5)
// instead of the nine gradients: reconstruction and the L/R average are linear, so reconstructing tau
// equals forming tau from reconstructed gradients up to rounding, with 6 fields instead of 9.
// Ghosts of tau follow the BC index map like those of G (reading A19).  At a face along d
//   tau_ad^f = 1/2 (L + R) of the fifth-order reconstructions   (= the symmetric 6-point formula)
//   u^f      = 1/2 (m_L / rho_L + m_R / rho_R)                   (velocity of the reconstructed state)
//   H        = (tau_xd, tau_yd, tau_zd, u . tau_d)^f,   r[1..4] += (H^+ - H^-) / dx.
#pragma once
#include <cuda.h>
#include "igr_common.cuh"

// field order inside the tau block: xx, xy, xz, yy, yz, zz
#define IGR_TAU_XX 0
#define IGR_TAU_XY 1
#define IGR_TAU_XZ 2
#define IGR_TAU_YY 3
#define IGR_TAU_YZ 4
#define IGR_TAU_ZZ 5

struct TauPtrs { float *t[6]; };             // t[0] == NULL: the source kernel does not write tau

struct ViscTileMaps {
    CUtensorMap q[3];      // 4-D maps (x, y, z, field) over rho, m (4 fields) of the three state buffers
    CUtensorMap tau;       // 4-D map over the first five tau fields (the in-plane faces never need tau_zz)
    bool valid;
};

namespace igr_visc {

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// left / right reconstruction at the face between stencil cells 2 | 3 (explicit rounding intrinsics:
// every inlined instance gives bitwise the same value)
template <int ORDER>
__device__ __forceinline__ void recon_lr(const float t[6], float &l, float &r)
{
    if (ORDER == 5) {
        l = __fmul_rn(2.f / 60.f, t[0]);
        l = __fmaf_rn(-13.f / 60.f, t[1], l);
        l = __fmaf_rn(47.f / 60.f, t[2], l);
        l = __fmaf_rn(27.f / 60.f, t[3], l);
        l = __fmaf_rn(-3.f / 60.f, t[4], l);
        r = __fmul_rn(-3.f / 60.f, t[1]);
        r = __fmaf_rn(27.f / 60.f, t[2], r);
        r = __fmaf_rn(47.f / 60.f, t[3], r);
        r = __fmaf_rn(-13.f / 60.f, t[4], r);
        r = __fmaf_rn(2.f / 60.f, t[5], r);
    } else {
        l = __fmul_rn(-1.f / 6.f, t[1]);
        l = __fmaf_rn(5.f / 6.f, t[2], l);
        l = __fmaf_rn(2.f / 6.f, t[3], l);
        r = __fmul_rn(2.f / 6.f, t[2]);
        r = __fmaf_rn(5.f / 6.f, t[3], r);
        r = __fmaf_rn(-1.f / 6.f, t[4], r);
    }
}

// 1/2 (L + R): the symmetric formula, coefficients (1, -8, 37, 37, -8, 1)/60 resp. (-1, 7, 7, -1)/12
template <int ORDER>
__device__ __forceinline__ float recon_mid(const float t[6])
{
    float v;
    if (ORDER == 5) {
        v = __fmul_rn(1.f / 60.f, __fadd_rn(t[0], t[5]));
        v = __fmaf_rn(-8.f / 60.f, __fadd_rn(t[1], t[4]), v);
        v = __fmaf_rn(37.f / 60.f, __fadd_rn(t[2], t[3]), v);
    } else {
        v = __fmul_rn(-1.f / 12.f, __fadd_rn(t[1], t[4]));
        v = __fmaf_rn(7.f / 12.f, __fadd_rn(t[2], t[3]), v);
    }
    return v;
}

// H at one face from the six stencil cells of (rho, mx, my, mz) and of (tau_xd, tau_yd, tau_zd)
template <int ORDER>
__device__ __forceinline__ void face(const float tq[4][6], const float tt[3][6], float H[4])
{
    float L[4], R[4];
#pragma unroll
    for (int f = 0; f < 4; ++f) recon_lr<ORDER>(tq[f], L[f], R[f]);
    const float il = __fmul_rn(0.5f, rcp_approx(L[0])), ir = __fmul_rn(0.5f, rcp_approx(R[0]));
    float e = 0.f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float uf = __fmaf_rn(R[1 + a], ir, __fmul_rn(L[1 + a], il));
        H[a] = recon_mid<ORDER>(tt[a]);
        e = (a == 0) ? __fmul_rn(uf, H[a]) : __fmaf_rn(uf, H[a], e);
    }
    H[3] = e;
}

// tau fields feeding the faces along d: (tau_xd, tau_yd, tau_zd)
__host__ __device__ constexpr int tau_field(int d, int a)
{
    return (d == 0) ? (a == 0 ? IGR_TAU_XX : (a == 1 ? IGR_TAU_XY : IGR_TAU_XZ))
         : (d == 1) ? (a == 0 ? IGR_TAU_XY : (a == 1 ? IGR_TAU_YY : IGR_TAU_YZ))
                    : (a == 0 ? IGR_TAU_XZ : (a == 1 ? IGR_TAU_YZ : IGR_TAU_ZZ));
}

}  // namespace igr_visc

struct ViscTileArgs {
    const void *q[5];      // current stage state (own-column reads for the z stencil; E only when fused)
    const float *tau;      // block of six padded fp32 fields, field stride g.np
    float *r[5];           // RHS rows: r[1..4] are read-modify-written (unfused) or read (fused)
    float inv_dx;
    int zc;                // planes per z-chunk (0: default)
    // fused with rows a5/a6: q_out = q_n + beta ((q_s - q_n) + dt (r + viscous part)); r is not written
    const void *qn[5];
    void *qout[5];         // must not alias q (q is read with its stencil halo); may alias qn
    float beta, dt, gamma;
    int read_qn;           // 0 in stage 1 (q_n == q_s)
    WaveResult *wave;      // stage 3: wave speed of q_out (may be NULL)
};

// returns 0 on success (message in `err` otherwise)
int visc_tile_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state, const float *tau,
                        ViscTileMaps *out, const char **err);
void launch_viscous_tile(const Grid &g, int storage, int order, bool fused, const CUtensorMap &qmap,
                         const CUtensorMap &tmap, ViscTileArgs a, cudaStream_t st);
