// igr_jacobi_blocked.cu -- row a3 of the hot path for sm_100a: NS (= n_jacobi, up to 5) warm-started
// Jacobi sweeps of
//     Sigma/rho - alpha div(grad(Sigma)/rho) = b          (eq. 9; A1-A3)
// temporally blocked: ONE pass over HBM reads rho, b, Sigma_old and writes Sigma_new after all NS
// sweeps (16 B per cell instead of 16 B per sweep).
//
// Design: 2.5-D streaming with a skewed pipeline of sweep levels.
// A CTA of 1024 threads owns a 32 x 32 column region = (32-2NS)^2 output columns + an NS-wide halo
// that is recomputed (the dependency cone of NS sweeps), and marches along z.  At step tau the plane
// p0 enters; level l+1 (l = 0..NS-1) advances its iterate on plane p0-1-l from level l's planes
// p0-2-l .. p0-l.  In-plane neighbours come from double-buffered shared-memory planes (one per
// level), the z neighbours and all seven stencil coefficients of the NS planes in flight live in
// registers (a compile-time rotated ring, so nothing is shifted).  One __syncthreads per plane.
// Ghost values of every iterate follow the BC index map at every sweep (wrap / clamp, reading A8):
// periodic directions are recomputed from wrapped data, clamp directions read the cell itself in
// place of its outside neighbour.
#include "igr_kernels.h"

namespace {

constexpr int R = 32;                       // region edge (threads per CTA = R*R)

struct Coef { float wxm, wxp, wym, wyp, wzp, dinv, b; };

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// index for rho: wrapped if periodic, else clamped to [-1, n] (keeps the first ghost layer, whose
// density enters the face weights; inflow ghosts differ from the clamp value)
__device__ __forceinline__ int rho_index(int i, int n, bool periodic)
{
    if (periodic) { i %= n; return i < 0 ? i + n : i; }
    return min(max(i, -1), n);
}

template <typename T, int NS>
__global__ void __launch_bounds__(R * R, 1)
k_jacobi_blocked(Grid g, const T *__restrict__ rho, const float *__restrict__ bsrc, const T *__restrict__ sin,
                 T *__restrict__ sout, float k2, int zc)
{
    constexpr int OT = R - 2 * NS;
    constexpr int P = R + 2;                 // padded plane pitch: a border of one cell, so that the
    constexpr int PP = P * (R + 2);          // four in-plane neighbours are at constant offsets
    extern __shared__ __align__(16) float jb_smem[];
    float (*RHO)[PP] = reinterpret_cast<float (*)[PP]>(jb_smem);                       // [2][PP]
    float (*SP)[2][PP] = reinterpret_cast<float (*)[2][PP]>(jb_smem + 2 * PP);          // [NS][2][PP]

    const int rx = threadIdx.x & 31, ry = threadIdx.x >> 5, pos = (ry + 1) * P + rx + 1;
    const int gi = blockIdx.x * OT - NS + rx, gj = blockIdx.y * OT - NS + ry;
    const int kz0 = blockIdx.z * zc, nkz = min(zc, g.nz - kz0);
    const bool per_x = g.bc[0] == 0, per_y = g.bc[2] == 0, per_z = g.bc[4] == 0;

    // Store mask of this thread for the iterate planes.  Ghost values follow the BC index map at
    // every sweep: a cell on a clamp boundary also writes its value into the neighbouring ghost
    // position, and threads at positions outside a clamped domain do not store at all.
    enum { ST_OWN = 1, ST_W = 2, ST_E = 4, ST_S = 8, ST_N = 16, ST_CORE = 32 };
    int mask = 0;
    {
        const bool in_x = per_x || (gi >= 0 && gi < g.nx), in_y = per_y || (gj >= 0 && gj < g.ny);
        if (in_x && in_y) {
            mask |= ST_OWN;
            if (!per_x && gi == 0) mask |= ST_W;
            if (!per_x && gi == g.nx - 1) mask |= ST_E;
            if (!per_y && gj == 0) mask |= ST_S;
            if (!per_y && gj == g.ny - 1) mask |= ST_N;
        }
        if (rx >= NS && rx < R - NS && ry >= NS && ry < R - NS && gi < g.nx && gj < g.ny) mask |= ST_CORE;
    }
    auto put = [&](float *plane, float v) {
        if (mask & ST_OWN) plane[pos] = v;
        if (mask & ST_W) plane[pos - 1] = v;
        if (mask & ST_E) plane[pos + 1] = v;
        if (mask & ST_S) plane[pos - P] = v;
        if (mask & ST_N) plane[pos + P] = v;
    };

    // element offsets fit 32 bits for every grid that fits the device memory
    const unsigned off_r = (unsigned)(rho_index(gi, g.nx, per_x) + g.gx) +
                           (unsigned)g.sy * (unsigned)(rho_index(gj, g.ny, per_y) + IGR_NG);
    const unsigned off_m = (unsigned)(map_index(gi, g.nx, g.bc[0]) + g.gx) +
                           (unsigned)g.sy * (unsigned)(map_index(gj, g.ny, g.bc[2]) + IGR_NG);
    const unsigned off_o = (unsigned)(gi + g.gx) + (unsigned)g.sy * (unsigned)(gj + IGR_NG);
    const unsigned usz = (unsigned)g.sz;

    auto load_plane = [&](int p, float &r0, float &b0, float &s0) {
        const unsigned zr = usz * (unsigned)(rho_index(p, g.nz, per_z) + IGR_NG);
        const unsigned zm = usz * (unsigned)(map_index(p, g.nz, g.bc[4]) + IGR_NG);
        r0 = ldf(rho + (off_r + zr));
        b0 = bsrc[off_m + zm];
        s0 = ldf(sin + (off_m + zm));
    };

    Coef C[NS];                              // ring: coefficient set of plane p lives in slot p mod NS
    float below[NS], centre[NS];             // own column: level-l iterate at planes c-1, c (c = p1 - l)
#pragma unroll
    for (int l = 0; l < NS; ++l) {
        C[l].wxm = C[l].wxp = C[l].wym = C[l].wyp = C[l].wzp = C[l].dinv = C[l].b = 0.f;
        below[l] = centre[l] = 0.f;
    }
    float rho1 = 1.f, b1 = 0.f, wz_prev = 0.f;
    for (int e = threadIdx.x; e < PP; e += R * R) {
        RHO[0][e] = 1.f; RHO[1][e] = 1.f;
#pragma unroll
        for (int l = 0; l < NS; ++l) { SP[l][0][e] = 0.f; SP[l][1][e] = 0.f; }
    }

    const int kfirst = kz0 - NS;             // first plane that enters; plane p <-> step p - kfirst
    const int nsteps = nkz + 2 * NS;         // output plane of step tau is kfirst + tau - NS
    const float k22 = 2.0f * k2;
    float rn0, bn0, sn0;
    load_plane(kfirst, rn0, bn0, sn0);
    __syncthreads();

    for (int base = 0; base < nsteps; base += NS) {
#pragma unroll
        for (int u = 0; u < NS; ++u) {
            const int tau = base + u;
            const int p0 = kfirst + tau, p1 = p0 - 1;
            const float rho0 = rn0, b0 = bn0, s0 = sn0;
            if (tau + 1 < nsteps) load_plane(p0 + 1, rn0, bn0, sn0);        // prefetch the next plane
            const int par0 = tau & 1, par1 = par0 ^ 1;                       // parity of planes p0 / p1
            RHO[par0][pos] = rho0;
            put(SP[0][par0], s0);

            // ---- coefficients of plane p1 (its densities were stored in the previous step).
            // Slot of plane p1 in the ring: (u - 1) mod NS (compile time); it held plane p1 - NS.
            const int slot1 = (u + NS - 1) % NS;
            const float wz_old = C[slot1].wzp;                               // W_z+ of plane p1 - NS
            {
                const float *rp = &RHO[par1][pos];
                Coef c;
                c.wxm = k22 * rcp_approx(rho1 + rp[-1]);
                c.wxp = k22 * rcp_approx(rho1 + rp[1]);
                c.wym = k22 * rcp_approx(rho1 + rp[-P]);
                c.wyp = k22 * rcp_approx(rho1 + rp[P]);
                c.wzp = k22 * rcp_approx(rho1 + rho0);
                c.dinv = rcp_approx(rcp_approx(rho1) + ((c.wxm + c.wxp) + (c.wym + c.wyp) + (wz_prev + c.wzp)));
                c.b = b1;
                wz_prev = c.wzp;                                              // W_z- of the next plane
                C[slot1] = c;
            }

            // ---- levels: level l+1 advances plane c = p1 - l
            float above = s0;                                                 // level-0 iterate at plane p0
#pragma unroll
            for (int l = 0; l < NS; ++l) {
                const int c = p1 - l;
                const int slot = (u + 2 * NS - 1 - l) % NS;                   // slot of plane c
                const int slot_m = (u + 2 * NS - 2 - l) % NS;                 // slot of plane c - 1
                const float wzm = (l == NS - 1) ? wz_old : C[slot_m].wzp;
                const float *sp = &SP[l][(par1 + l) & 1][pos];                // plane c of level l
                const float ctr = centre[l];
                const float dn = (!per_z && c == 0) ? ctr : below[l];
                const float up = (!per_z && c == g.nz - 1) ? ctr : above;
                float acc = C[slot].b;
                acc = fmaf(C[slot].wxm, sp[-1], acc);
                acc = fmaf(C[slot].wxp, sp[1], acc);
                acc = fmaf(C[slot].wym, sp[-P], acc);
                acc = fmaf(C[slot].wyp, sp[P], acc);
                acc = fmaf(wzm, dn, acc);
                acc = fmaf(C[slot].wzp, up, acc);
                const float fresh = acc * C[slot].dinv;                       // level l+1 at plane c
                below[l] = ctr;
                centre[l] = above;
                above = fresh;
                if (l + 1 < NS) put(SP[l + 1][(par1 + l) & 1], fresh);       // plane c of level l+1
            }
            // `above` now holds the level-NS iterate at plane p1 - (NS - 1) = p0 - NS
            const int ko = p0 - NS;
            if ((mask & ST_CORE) && ko >= kz0 && ko < kz0 + nkz) stf(sout + (off_o + usz * (unsigned)(ko + IGR_NG)), above);
            rho1 = rho0; b1 = b0;
            __syncthreads();
        }
    }
}

}  // namespace

int jacobi_blocked_zc(const Grid &g, int ns)
{
    const int ot = R - 2 * ns;
    const long long cols = (long long)((g.nx + ot - 1) / ot) * ((g.ny + ot - 1) / ot);
    long long nch = (2LL * 148 + cols - 1) / cols;          // aim at >= 2 waves of 148 CTAs
    if (nch < 1) nch = 1;
    int zc = (int)((g.nz + nch - 1) / nch);
    if (zc < 8 * ns) zc = 8 * ns;                           // keep the 2 NS warm-up planes <= 25 %
    if (zc > g.nz) zc = g.nz;
    return zc;
}

template <typename T>
static void launch_ns(const Grid &g, int ns, const void *rho, const float *b, const void *sin, void *sout,
                      float k2, cudaStream_t st)
{
    const int ot = R - 2 * ns, zc = jacobi_blocked_zc(g, ns);
    dim3 grid((g.nx + ot - 1) / ot, (g.ny + ot - 1) / ot, (g.nz + zc - 1) / zc);
    const int smem = (2 + 2 * ns) * (R + 2) * (R + 2) * 4;
#define IGR_JB(NSV)                                                                                      \
    do {                                                                                                 \
        static bool configured = false;                                                                  \
        if (!configured) {                                                                               \
            cudaFuncSetAttribute(k_jacobi_blocked<T, NSV>, cudaFuncAttributeMaxDynamicSharedMemorySize,  \
                                 (2 + 2 * NSV) * (R + 2) * (R + 2) * 4);                                 \
            configured = true;                                                                           \
        }                                                                                                \
        k_jacobi_blocked<T, NSV><<<grid, R * R, smem, st>>>(g, (const T *)rho, b, (const T *)sin,        \
                                                           (T *)sout, k2, zc);                           \
    } while (0)
    switch (ns) {
    case 1: IGR_JB(1); break;
    case 2: IGR_JB(2); break;
    case 3: IGR_JB(3); break;
    case 4: IGR_JB(4); break;
    default: IGR_JB(5); break;
    }
#undef IGR_JB
}

// ns in 1..5 sweeps in one pass; sig_in and sig_out must differ
void launch_jacobi_blocked(const Grid &g, int storage, int ns, const void *rho, const float *b,
                           const void *sig_in, void *sig_out, float k2, cudaStream_t st)
{
    if (storage == 0) launch_ns<float>(g, ns, rho, b, sig_in, sig_out, k2, st);
    else if (storage == 1) launch_ns<__half>(g, ns, rho, b, sig_in, sig_out, k2, st);
    else launch_ns<__nv_bfloat16>(g, ns, rho, b, sig_in, sig_out, k2, st);
}
