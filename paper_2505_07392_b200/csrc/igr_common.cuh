// igr_common.cuh -- shared device/host definitions of libigr (B200, sm_100a).
//
// Data layout in HBM: every field is a padded SoA array
//   f[(k + NG) * PY + (j + NG)][i + GX],   pitch PX elements, x fastest,
// NG = 3 ghost layers in y and z, GX = 32 bytes of ghost/padding in x (8 fp32 / 16 half elements,
// of which the 3 next to the interior are the ghost cells), PX = round_up(nx + 2 GX, 32 bytes).
// Interior rows therefore start 32-byte aligned (sector aligned) and all TMA strides are
// multiples of 16 bytes.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <cuda_bf16.h>
#include <stdint.h>

#define IGR_NG 3

struct Grid {
    int nx, ny, nz;        // interior cells
    int gx;                // x ghost/padding elements (>= 3)
    int px, py, pz;        // padded extents (elements)
    long long sy, sz;      // strides in elements: sy = px, sz = px * py
    long long np;          // px * py * pz
    int bc[6];             // IGR_BC_* per face
    int wk0, wk1;          // planes [wk0, wk1) that enter the wave-speed reduction (default: all; slabs: owned)
    __host__ __device__ long long idx(int i, int j, int k) const {   // interior-relative indices
        return (long long)(i + gx) + sy * (long long)(j + IGR_NG) + sz * (long long)(k + IGR_NG);
    }
};

// index map of the boundary conditions (reading A8): periodic -> wrap, otherwise clamp
__host__ __device__ inline int map_index(int i, int n, int bc_lo)
{
    if (i >= 0 && i < n) return i;
    if (bc_lo == 0) { int m = i % n; return m < 0 ? m + n : m; }
    return i < 0 ? 0 : n - 1;
}

// Domain decomposition (igr.h IGR_BC_EXTERNAL; reading A20): a ghost cell beyond an external face
// along any of its out-of-range axes is the neighbouring sub-domain's (or an edge/corner cell no stencil
// reads): the halo kernels never write it.  Everywhere else an external face acts like a clamp.
constexpr int kBcExternal = 3;
__host__ __device__ inline bool ghost_is_external(const Grid &g, int i, int j, int k)
{
    return (i < 0 && g.bc[0] == kBcExternal) || (i >= g.nx && g.bc[1] == kBcExternal) ||
           (j < 0 && g.bc[2] == kBcExternal) || (j >= g.ny && g.bc[3] == kBcExternal) ||
           (k < 0 && g.bc[4] == kBcExternal) || (k >= g.nz && g.bc[5] == kBcExternal);
}

// ---- storage <-> fp32 (FP16 storage, FP32 compute)
__device__ __forceinline__ float ldf(const float *p) { return *p; }
__device__ __forceinline__ float ldf(const __half *p) { return __half2float(*p); }
__device__ __forceinline__ float ldf(const __nv_bfloat16 *p) { return __bfloat162float(*p); }
__device__ __forceinline__ void stf(float *p, float v) { *p = v; }
__device__ __forceinline__ void stf(__half *p, float v) { *p = __float2half_rn(v); }
__device__ __forceinline__ void stf(__nv_bfloat16 *p, float v) { *p = __float2bfloat16_rn(v); }

struct StagePtrs {            // device pointers of one state buffer (5 padded fields; 7 with two fluids)
    void *f[7];
};

// inflow description of one face, device resident (weights precomputed on the host in fp64)
struct InflowFace {
    const float *weight;      // [n1][n0] blend weight w in [0,1] per transverse cell (NULL: none)
    const float *fixed;       // [n1][n0][5] fixed conserved state of the winning patch
    int n0, n1;               // transverse extents
};

struct BcDesc {
    InflowFace inflow[6];
};

// fp64 mode (IGR_STORE_F64): inflow tables in double, wave result in 64 bits
struct Inflow64 {
    const double *weight[6];  // [n1][n0] blend weight per transverse cell (NULL: none)
    const double *fixed[6];   // [n1][n0][5]
    int n0[6], n1[6];
};
struct WaveResult64 {
    unsigned long long max_bits;   // double bits of the maximum wave speed (non-negative)
    unsigned int nonfinite;
};

// ordered-int encoding of non-negative floats for atomicMax
struct WaveResult {
    unsigned int max_bits;    // float bits of the maximum wave speed (non-negative)
    unsigned int nonfinite;   // != 0 if any cell produced a non-finite value
};

// max_d |u_d| + c of one cell with IEEE division and square root (rows a5/a6); sets `bad` instead of
// returning a non-finite value
__device__ __forceinline__ float wavespeed_of(float rho, float mx, float my, float mz, float E,
                                              float gamma, bool &bad)
{
    // explicit rounding intrinsics: every inlined instance gives bitwise the same value
    const float ir = __fdiv_rn(1.0f, rho);
    float m2 = __fmul_rn(mx, mx);
    m2 = __fmaf_rn(my, my, m2);
    m2 = __fmaf_rn(mz, mz, m2);
    const float p = __fmul_rn(gamma - 1.0f, __fmaf_rn(__fmul_rn(-0.5f, ir), m2, E));
    const float c = __fsqrt_rn(__fmul_rn(__fmul_rn(gamma, p), ir));
    const float v = __fmaf_rn(fmaxf(fabsf(mx), fmaxf(fabsf(my), fabsf(mz))), fabsf(ir), c);
    // non-finite (NaN/Inf, or sqrt of a negative) is reported, never repaired (reading A10)
    if (!(v <= 3.0e38f)) { bad = true; return 0.f; }
    return v;
}

// the same for two fluids (reading A21): q = (a1 rho1, a2 rho2, m, E, a1), c^2 = (1 + 1/Gamma) p / rho,
// Gamma = a1 k1 + (1 - a1) k2, k_i = 1/(gamma_i - 1)
__device__ __forceinline__ float wavespeed_of2(const float *q, float k1, float k2, bool &bad)
{
    const float rho = __fadd_rn(q[0], q[1]);
    const float ir = __fdiv_rn(1.0f, rho);
    float m2 = __fmul_rn(q[2], q[2]);
    m2 = __fmaf_rn(q[3], q[3], m2);
    m2 = __fmaf_rn(q[4], q[4], m2);
    const float g1 = __fdiv_rn(1.0f, __fmaf_rn(q[6], k1 - k2, k2));
    const float p = __fmul_rn(g1, __fmaf_rn(__fmul_rn(-0.5f, ir), m2, q[5]));
    const float c = __fsqrt_rn(__fmul_rn(__fmul_rn(__fadd_rn(1.0f, g1), p), ir));
    const float v = __fmaf_rn(fmaxf(fabsf(q[2]), fmaxf(fabsf(q[3]), fabsf(q[4]))), fabsf(ir), c);
    if (!(v <= 3.0e38f)) { bad = true; return 0.f; }
    return v;
}

#define IGR_CUDA_OK(call)                                                                          \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) return s->fail(IGR_ERR_CUDA, #call, e_);                            \
    } while (0)
