// igr_source_tma.cu -- row a2 of the hot path for sm_100a, TMA-staged form (round 2):
//     b = alpha ( tr((grad u)^2) + (tr grad u)^2 ),   G_ab = d u_a / d x_b by second-order central differences of
// the cell-centred velocity u = m / rho            (eq. 9, footnote L252; L132; Alg. 1).
//
// Same 2.5-D plan as k_source (igr_kernels.cu): a CTA owns a 32 x 8 column of cells and marches along z; each cell's
// velocity is formed once (one reciprocal) and shared with its in-plane neighbours through shared memory, the z
// neighbours are registers.  What changed: the raw planes of (rho, m_x, m_y, m_z) with their one-cell halo arrive
// by TMA (four 3-D boxes per plane issued by one elected lane, mbarrier ring, three planes ahead) instead of by
// per-thread global loads -- no address arithmetic, no separate sector-sized loads for the 80 halo cells of the
// tile -- and the nine differences stay undivided (1/(2 dx)^2 goes into the factor of the sum).  The ncu profile of
// k_source showed 108 instructions per cell at 68 % issue utilisation for 20 bytes per cell: issue-bound at 0.68 of
// the HBM ceiling.  The stress fields of the viscous variant stay with k_source.
#include "igr_kernels.h"
#include "igr_tma.cuh"

#include <cuda.h>

namespace {

constexpr int TX = 32, TY = 8;
constexpr int NSLOT = 4;                    // raw planes: one being consumed, three in flight
constexpr int PW = TX + 2, PH = TY + 2, PN = PW * PH;      // velocity planes with a one-cell halo

template <typename T>
struct Box {
    static constexpr int HX = 16 / (int)sizeof(T);          // x halo of the box in elements: 16 bytes (alignment)
    static constexpr int BX = TX + 2 * HX, BY = TY + 2;
    static constexpr int PE = BX * BY;                      // elements of one field
    static constexpr int FBYTES = (PE * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int SLOT = 4 * FBYTES;
};

__device__ __forceinline__ float rcp_fast(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <typename T>
__global__ void __launch_bounds__(TX * TY)
k_source_tma(const __grid_constant__ CUtensorMap m0, const __grid_constant__ CUtensorMap m1,
             const __grid_constant__ CUtensorMap m2, const __grid_constant__ CUtensorMap m3, Grid g,
             float *__restrict__ b, float coef, int zc)
{
    using BXT = Box<T>;
    extern __shared__ __align__(1024) unsigned char ss[];
    float (*U)[3][PN] = reinterpret_cast<float (*)[3][PN]>(ss + NSLOT * BXT::SLOT);       // [3 planes][3][PN]
    uint64_t *full = reinterpret_cast<uint64_t *>(ss + NSLOT * BXT::SLOT + 3 * 3 * PN * 4);

    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int kz0 = blockIdx.z * zc, nkz = min(zc, g.nz - kz0);
    const bool valid = (x0 + tx < g.nx) && (y0 + ty < g.ny);
    const int wu = __shfl_sync(0xffffffffu, tid >> 5, 0);

    // plane p <-> cell plane kz0 - 1 + p (p = 0 .. nkz + 1)
    const int cx = g.gx + x0 - BXT::HX, cy = IGR_NG + y0 - 1, cz = IGR_NG + kz0 - 1;
    auto issue = [&](int p, int slot) {
        unsigned char *dst = ss + slot * BXT::SLOT;
        igr_tma::mbar_expect_tx(&full[slot], 4 * BXT::PE * (int)sizeof(T));
        igr_tma::tma_load_3d(dst, &m0, cx, cy, cz + p, &full[slot]);
        igr_tma::tma_load_3d(dst + BXT::FBYTES, &m1, cx, cy, cz + p, &full[slot]);
        igr_tma::tma_load_3d(dst + 2 * BXT::FBYTES, &m2, cx, cy, cz + p, &full[slot]);
        igr_tma::tma_load_3d(dst + 3 * BXT::FBYTES, &m3, cx, cy, cz + p, &full[slot]);
    };
    auto elect_one = []() {
        uint32_t pred;
        asm volatile("{\n .reg .pred P;\n elect.sync _|P, 0xffffffff;\n selp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
        return pred != 0;
    };
    const int n_planes = nkz + 2;
    if (tid == 0) {
        for (int s = 0; s < NSLOT; ++s) igr_tma::mbar_init(&full[s], 1);
        igr_tma::fence_init();
    }
    __syncthreads();
    if (wu == 0 && elect_one())
        for (int p = 0; p < NSLOT && p < n_planes; ++p) issue(p, p);

    // own cell and (first 80 threads) one cell of the tile's halo ring, as positions in the box and in a velocity plane
    const int own_b = (ty + 1) * BXT::BX + BXT::HX + tx, own_u = (ty + 1) * PW + tx + 1;
    int halo_b = -1, halo_u = 0;
    if (tid < 2 * TX + 2 * TY) {
        int hx, hy;
        if (tid < 2 * TX) { hx = tid & 31; hy = (tid >> 5) ? TY : -1; }
        else { const int t = tid - 2 * TX; hy = t % TY; hx = (t / TY) ? TX : -1; }
        halo_b = (hy + 1) * BXT::BX + BXT::HX + hx;
        halo_u = (hy + 1) * PW + hx + 1;
    }
    // raw plane in `slot` -> velocities into velocity plane `up`; returns the own cell's velocity
    auto velocities = [&](int slot, int up, float v[3]) {
        const T *raw = reinterpret_cast<const T *>(ss + slot * BXT::SLOT);
        constexpr int FE = BXT::FBYTES / (int)sizeof(T);
        const float ir = rcp_fast(ldf(raw + own_b));
        v[0] = ldf(raw + FE + own_b) * ir; v[1] = ldf(raw + 2 * FE + own_b) * ir; v[2] = ldf(raw + 3 * FE + own_b) * ir;
        U[up][0][own_u] = v[0]; U[up][1][own_u] = v[1]; U[up][2][own_u] = v[2];
        if (halo_b >= 0) {
            const float hr = rcp_fast(ldf(raw + halo_b));
            U[up][0][halo_u] = ldf(raw + FE + halo_b) * hr;
            U[up][1][halo_u] = ldf(raw + 2 * FE + halo_b) * hr;
            U[up][2][halo_u] = ldf(raw + 3 * FE + halo_b) * hr;
        }
    };

    // prologue: planes 0 (cells kz0 - 1: only the own column is needed) and 1 (cells kz0)
    float dn[3], ce[3], up[3];
    igr_tma::mbar_wait(&full[0], 0);
    velocities(0, 2, dn);
    igr_tma::mbar_wait(&full[1], 0);
    velocities(1, 0, ce);
    __syncthreads();                                            // raw slots 0 and 1 are free, plane 0 of U is complete
    if (wu == 0 && elect_one()) {
        igr_tma::fence_async();
        for (int p = NSLOT; p < NSLOT + 2 && p < n_planes; ++p) issue(p, p - NSLOT);
    }

    unsigned slot = 2, phase = 0, uc = 0;                       // raw slot of plane t + 2; velocity plane of cell plane k
    unsigned id = (unsigned)(min(x0 + tx, g.nx - 1) + g.gx) + (unsigned)g.sy * (unsigned)(min(y0 + ty, g.ny - 1) + IGR_NG) +
                  (unsigned)g.sz * (unsigned)(kz0 + IGR_NG);
    // (three plane steps per loop trip, or a minimum of 4 / 6 CTAs per SM, were measured slower: 4.5 / 4.3 vs 4.25 ms)
    for (int t = 0; t < nkz; ++t) {
        const unsigned un = uc == 2 ? 0u : uc + 1u;              // velocity plane of cell plane k + 1
        igr_tma::mbar_wait(&full[slot], phase);
        velocities((int)slot, (int)un, up);
        __syncthreads();                                        // the only barrier of the step
        if (wu == 0 && t + 2 + NSLOT < n_planes && elect_one()) {      // the raw slot just read is free again
            igr_tma::fence_async();
            issue(t + 2 + NSLOT, (int)slot);
        }
        const float (*P)[PN] = U[uc];
        float G[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            G[a][0] = P[a][own_u + 1] - P[a][own_u - 1];
            G[a][1] = P[a][own_u + PW] - P[a][own_u - PW];
            G[a][2] = up[a] - dn[a];
        }
        const float tr = G[0][0] + G[1][1] + G[2][2];
        const float trsq = G[0][0] * G[0][0] + G[1][1] * G[1][1] + G[2][2] * G[2][2] +
                           2.0f * (G[0][1] * G[1][0] + G[0][2] * G[2][0] + G[1][2] * G[2][1]);
        if (valid) b[id] = coef * (trsq + tr * tr);
        id += (unsigned)g.sz;
#pragma unroll
        for (int a = 0; a < 3; ++a) { dn[a] = ce[a]; ce[a] = up[a]; }
        uc = un;
        if (++slot == NSLOT) { slot = 0; phase ^= 1u; }
    }
}

template <typename T>
void launch_t(const Grid &g, const SourceMaps &m, float *b, float coef, cudaStream_t st)
{
    using BXT = Box<T>;
    constexpr int smem = NSLOT * BXT::SLOT + 3 * 3 * PN * 4 + NSLOT * 8 + 8;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_source_tma<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        configured = true;
    }
    // z chunks: enough CTAs for several waves, at least 32 planes each (two warm-up planes per chunk)
    const long long cols = (long long)((g.nx + TX - 1) / TX) * ((g.ny + TY - 1) / TY);
    long long nch = (8LL * 148 * 4 + cols - 1) / cols;
    if (nch < 1) nch = 1;
    int zc = (int)((g.nz + nch - 1) / nch);
    if (zc < 32) zc = 32;
    if (zc > g.nz) zc = g.nz;
    dim3 grid((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + zc - 1) / zc);
    k_source_tma<T><<<grid, TX * TY, smem, st>>>(m.f[0], m.f[1], m.f[2], m.f[3], g, b, coef, zc);
}

}  // namespace

// 3-D maps of (rho, m_x, m_y, m_z) with boxes of (32 + 32 bytes) x 10 x 1
int source_make_maps(const Grid &g, int storage, void *const f[4], SourceMaps *out)
{
    out->valid = false;
    if (!igr_tma::get_encode()) return 1;
    const size_t es = storage == 0 ? 4 : 2;
    for (int c = 0; c < 4; ++c) {
        cuuint64_t dims[3] = { (cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz };
        cuuint64_t strides[2] = { (cuuint64_t)g.px * es, (cuuint64_t)g.px * g.py * es };
        cuuint32_t box[3] = { (cuuint32_t)(TX + 32 / es), TY + 2, 1 };
        if (!igr_tma::encode(&out->f[c], igr_tma::data_type(storage), 3, f[c], dims, strides, box)) return 2;
    }
    out->valid = true;
    return 0;
}

void launch_source_tma(const Grid &g, int storage, const SourceMaps &m, float *b, float alpha, float inv2dx,
                       cudaStream_t st)
{
    const float coef = alpha * inv2dx * inv2dx;
    if (storage == 0) launch_t<float>(g, m, b, coef, st);
    else if (storage == 1) launch_t<__half>(g, m, b, coef, st);
    else launch_t<__nv_bfloat16>(g, m, b, coef, st);
}
