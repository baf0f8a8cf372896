// igr_kernels.cu -- boundary/halo, source, simple Jacobi sweep, simple RHS, RK update and the
// wave-speed reduction of libigr (sm_100a).  Citations are PAPER.md lines; readings are DESIGN.md's.
// The tiled/TMA RHS kernel and the temporally blocked Jacobi kernel live in their own files.
#include "igr_kernels.h"
#include "igr_viscous.cuh"

#define IGR_STORE_F32 0
#define IGR_STORE_F16 1
#define IGR_STORE_BF16 2

#define DISPATCH_STORAGE(storage, ...)                                                             \
    do {                                                                                           \
        if ((storage) == IGR_STORE_F32) { typedef float T; __VA_ARGS__; }                          \
        else if ((storage) == IGR_STORE_F16) { typedef __half T; __VA_ARGS__; }                    \
        else { typedef __nv_bfloat16 T; __VA_ARGS__; }                                             \
    } while (0)

static inline unsigned int blocks_for(long long n, int threads, long long cap = 1 << 20)
{
    long long b = (n + threads - 1) / threads;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned int)b;
}

// ------------------------------------------------------------------------------ pack / unpack
template <typename T>
__global__ void k_unpack(Grid g, const float *__restrict__ user, T *__restrict__ field, int k0, int nk)
{
    long long n = (long long)nk * g.ny * g.nx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx);
        long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        stf(field + g.idx(i, j, k0 + k), user[t]);
    }
}

template <typename T>
__global__ void k_pack(Grid g, const T *__restrict__ field, float *__restrict__ user, int k0, int nk)
{
    long long n = (long long)nk * g.ny * g.nx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx);
        long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        user[t] = ldf(field + g.idx(i, j, k0 + k));
    }
}

template <typename T>
__global__ void k_pack_padded(Grid g, const T *__restrict__ field, float *__restrict__ user, int k0, int nk)
{
    const int wx = g.nx + 2 * IGR_NG, wy = g.ny + 2 * IGR_NG;
    long long n = (long long)nk * wy * wx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % wx);
        long long r = t / wx;
        int j = (int)(r % wy), k = (int)(r / wy);
        user[t] = ldf(field + g.idx(i - IGR_NG, j - IGR_NG, k0 + k - IGR_NG));
    }
}

void launch_unpack_field(const Grid &g, int storage, const float *user, void *field, int k0, int nk,
                         cudaStream_t st)
{
    long long n = (long long)nk * g.ny * g.nx;
    DISPATCH_STORAGE(storage, k_unpack<T><<<blocks_for(n, 256), 256, 0, st>>>(g, user, (T *)field, k0, nk));
}

void launch_pack_field(const Grid &g, int storage, const void *field, float *user, int k0, int nk,
                       cudaStream_t st)
{
    long long n = (long long)nk * g.ny * g.nx;
    DISPATCH_STORAGE(storage, k_pack<T><<<blocks_for(n, 256), 256, 0, st>>>(g, (const T *)field, user, k0, nk));
}

void launch_unpack_f32(const Grid &g, const float *user, float *field, int k0, int nk, cudaStream_t st)
{
    launch_unpack_field(g, IGR_STORE_F32, user, field, k0, nk, st);
}

void launch_pack_f32(const Grid &g, const float *field, float *user, int k0, int nk, cudaStream_t st)
{
    launch_pack_field(g, IGR_STORE_F32, field, user, k0, nk, st);
}

void launch_pack_padded(const Grid &g, int storage, const void *field, float *user, int k0, int nk,
                        cudaStream_t st)
{
    long long n = (long long)nk * (g.ny + 2 * IGR_NG) * (g.nx + 2 * IGR_NG);
    DISPATCH_STORAGE(storage,
                     k_pack_padded<T><<<blocks_for(n, 256), 256, 0, st>>>(g, (const T *)field, user, k0, nk));
}

// ------------------------------------------------------------------------------ a1: halo / BC
// The paper gives no boundary conditions; BASELINE.json names periodic, extrapolation outflow and
// fixed-state inflow patches.  Reading A8: every ghost cell is a copy of the interior cell given by
// the per-axis index map (wrap / clamp), blended towards the fixed patch state on inflow faces.
// All ghosts read interior cells only, so one launch covers the three slabs (no ordering).
struct GhostCell { int i, j, k; bool valid; };

// (unsigned 32-bit arithmetic: the ghost cells of any grid that fits the device number far below 2^32, and a
// 64-bit division costs five times a 32-bit one; the halo kernels were spending their time here)
__device__ __forceinline__ GhostCell decode_ghost(const Grid &g, long long t64)
{
    const unsigned wx = g.nx + 2 * IGR_NG, wy = g.ny + 2 * IGR_NG;
    const unsigned nZ = 2u * IGR_NG * wy * wx;                   // full padded planes below/above
    const unsigned nY = (unsigned)g.nz * 2u * IGR_NG * wx;       // rows in front/behind, interior k
    const unsigned nX = (unsigned)g.nz * (unsigned)g.ny * 2u * IGR_NG;   // columns left/right, interior j, k
    unsigned t = (unsigned)t64;
    GhostCell c;
    c.valid = true;
    if (t < nZ) {
        const unsigned r = t / wx, i = t - r * wx, kk = r / wy, j = r - kk * wy;
        c.i = (int)i - IGR_NG; c.j = (int)j - IGR_NG; c.k = kk < IGR_NG ? (int)kk - IGR_NG : g.nz + ((int)kk - IGR_NG);
    } else if (t < nZ + nY) {
        t -= nZ;
        const unsigned r = t / wx, i = t - r * wx, k = r / (2u * IGR_NG), jj = r - k * (2u * IGR_NG);
        c.k = (int)k;
        c.i = (int)i - IGR_NG; c.j = jj < IGR_NG ? (int)jj - IGR_NG : g.ny + ((int)jj - IGR_NG);
    } else if (t < nZ + nY + nX) {
        t -= nZ + nY;
        const unsigned r = t / (2u * IGR_NG), ii = t - r * (2u * IGR_NG), k = r / (unsigned)g.ny, j = r - k * (unsigned)g.ny;
        c.j = (int)j; c.k = (int)k;
        c.i = ii < IGR_NG ? (int)ii - IGR_NG : g.nx + ((int)ii - IGR_NG);
    } else {
        c.valid = false; c.i = c.j = c.k = 0;
    }
    return c;
}

__host__ __device__ inline long long ghost_count(const Grid &g)
{
    const long long wx = g.nx + 2 * IGR_NG, wy = g.ny + 2 * IGR_NG;
    return 2LL * IGR_NG * wy * wx + (long long)g.nz * 2 * IGR_NG * wx + (long long)g.nz * g.ny * 2 * IGR_NG;
}

template <typename T>
__global__ void k_halo_q(Grid g, StagePtrs q, BcDesc bc, int nf)
{
    const long long n = ghost_count(g);
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        GhostCell c = decode_ghost(g, t);
        if (ghost_is_external(g, c.i, c.j, c.k)) continue;
        const long long dst = g.idx(c.i, c.j, c.k);
        const long long src = g.idx(map_index(c.i, g.nx, g.bc[0]), map_index(c.j, g.ny, g.bc[2]),
                                    map_index(c.k, g.nz, g.bc[4]));
        // inflow: first out-of-range axis (x, y, z order) whose face is an inflow face
        float w = 0.f;
        const float *fixed = nullptr;
        const int idx[3] = { c.i, c.j, c.k }, nn[3] = { g.nx, g.ny, g.nz };
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int face = idx[a] < 0 ? 2 * a : (idx[a] >= nn[a] ? 2 * a + 1 : -1);
            if (face < 0 || fixed != nullptr) continue;
            const InflowFace &f = bc.inflow[face];
            if (f.weight == nullptr) continue;
            int t0 = (a == 0) ? idx[1] : idx[0];
            int t1 = (a == 2) ? idx[1] : idx[2];
            if (t0 < 0 || t0 >= f.n0 || t1 < 0 || t1 >= f.n1) continue;   // edge/corner ghosts: never read
            float ww = f.weight[(long long)t1 * f.n0 + t0];
            if (ww > 0.f) { w = ww; fixed = f.fixed + ((long long)t1 * f.n0 + t0) * nf; }
        }
#pragma unroll
        for (int cmp = 0; cmp < 7; ++cmp) {
            if (cmp >= nf) break;
            T *fld = (T *)q.f[cmp];
            float v = ldf(fld + src);
            if (fixed != nullptr) v = (w >= 1.f) ? fixed[cmp] : v + w * (fixed[cmp] - v);
            stf(fld + dst, v);
        }
    }
}

template <typename T>
__global__ void k_halo_sigma(Grid g, T *__restrict__ sig)
{
    // Sigma ghosts: wrap on periodic faces, clamp on every other face (homogeneous Neumann, A8)
    const long long n = ghost_count(g);
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        GhostCell c = decode_ghost(g, t);
        if (ghost_is_external(g, c.i, c.j, c.k)) continue;
        const long long src = g.idx(map_index(c.i, g.nx, g.bc[0]), map_index(c.j, g.ny, g.bc[2]),
                                    map_index(c.k, g.nz, g.bc[4]));
        sig[g.idx(c.i, c.j, c.k)] = sig[src];
    }
}

// ghosts of `nf` derived fp32 fields (field stride g.np) by the index map alone: one launch
__global__ void k_halo_fields(Grid g, float *__restrict__ base, int nf)
{
    const long long n = ghost_count(g);
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        GhostCell c = decode_ghost(g, t);
        if (ghost_is_external(g, c.i, c.j, c.k)) continue;
        const long long src = g.idx(map_index(c.i, g.nx, g.bc[0]), map_index(c.j, g.ny, g.bc[2]),
                                    map_index(c.k, g.nz, g.bc[4]));
        const long long dst = g.idx(c.i, c.j, c.k);
        for (int f = 0; f < nf; ++f) base[f * g.np + dst] = base[f * g.np + src];
    }
}

void launch_halo_fields(const Grid &g, float *base, int nf, cudaStream_t st)
{
    long long n = ghost_count(g);
    k_halo_fields<<<blocks_for(n, 256, 148 * 16), 256, 0, st>>>(g, base, nf);
}

void launch_halo_q(const Grid &g, int storage, StagePtrs q, const BcDesc &bc, int nf, cudaStream_t st)
{
    long long n = ghost_count(g);
    DISPATCH_STORAGE(storage, k_halo_q<T><<<blocks_for(n, 256, 148 * 16), 256, 0, st>>>(g, q, bc, nf));
}

// two fluids: mixture density rho = a1 rho1 + a2 rho2 of EVERY cell of the padded array (ghosts included: the
// face weights of the Sigma equation read the first ghost layer), as one more fp32 field
__global__ void k_rho_total(const float *__restrict__ r1, const float *__restrict__ r2, float *__restrict__ out,
                            long long n)
{
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        out[t] = __fadd_rn(r1[t], r2[t]);
}

void launch_rho_total(const Grid &g, const float *r1, const float *r2, float *out, cudaStream_t st)
{
    k_rho_total<<<blocks_for(g.np, 256, 148 * 16), 256, 0, st>>>(r1, r2, out, g.np);
}

void launch_halo_sigma(const Grid &g, int storage, void *sig, cudaStream_t st)
{
    long long n = ghost_count(g);
    DISPATCH_STORAGE(storage, k_halo_sigma<T><<<blocks_for(n, 256, 148 * 16), 256, 0, st>>>(g, (T *)sig));
}

// ------------------------------------------------------------------------------ a2: source
// b = alpha ( tr((grad u)^2) + (tr grad u)^2 )  -- the side of eq. (9) that carries alpha (L127,
// footnote L252) with second-order central differences of the cell-centred velocity u = m/rho
// (L132; Alg. 1).  G_ab = d u_a / d x_b.
// Streaming form: a CTA owns a 32 x 8 column of cells and marches along z.  Each cell's velocity is
// computed once (one reciprocal per cell) and shared: in-plane neighbours through a ring of five
// shared-memory planes with a one-cell halo (two planes enter per barrier), z neighbours in registers.
// 4 loads + 1 store per cell.
constexpr int SRC_TX = 32, SRC_TY = 8, SRC_ZC = 128;

// GRAD: the same gradients also give the viscous stress tau (eq. 5; NEXT-1, igr_viscous.cuh), stored
// as six fp32 fields; mu2 = 2 mu, lam2 = zeta - 2 mu / 3.
template <typename T, bool GRAD>
__global__ void __launch_bounds__(SRC_TX * SRC_TY) k_source(Grid g, StagePtrs q, float *__restrict__ b,
                                                            float alpha, float inv2dx, TauPtrs tp, float mu,
                                                            float lam2)
{
    constexpr int PW = SRC_TX + 2, PH = SRC_TY + 2, PN = PW * PH;
    constexpr int NB = 5;                                    // plane buffers: two planes per barrier
    __shared__ float U[NB][3][PN];
    const T *rho = (const T *)q.f[0];
    const T *m[3] = { (const T *)q.f[1], (const T *)q.f[2], (const T *)q.f[3] };
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5, tid = threadIdx.x;
    const int x0 = blockIdx.x * SRC_TX, y0 = blockIdx.y * SRC_TY;
    const int kz0 = blockIdx.z * SRC_ZC, nkz = min(SRC_ZC, g.nz - kz0);
    // clamp the column into the padded array (columns beyond the domain compute unused values)
    const int i = min(x0 + tx, g.nx), j = min(y0 + ty, g.ny);
    const bool valid = (x0 + tx < g.nx) && (y0 + ty < g.ny);
    const unsigned usz = (unsigned)g.sz;
    const unsigned col = (unsigned)(i + g.gx) + (unsigned)g.sy * (unsigned)(j + IGR_NG);
    const int own = (ty + 1) * PW + tx + 1;
    // halo ring of the tile (2*32 + 2*8 cells): handled by the first 80 threads
    int hpos = -1; unsigned hcol = 0;
    if (tid < 2 * SRC_TX + 2 * SRC_TY) {
        int hx, hy;
        if (tid < 2 * SRC_TX) { hx = tid & 31; hy = (tid >> 5) ? SRC_TY : -1; }
        else { const int t = tid - 2 * SRC_TX; hy = t % SRC_TY; hx = (t / SRC_TY) ? SRC_TX : -1; }
        const int hi = min(max(x0 + hx, -1), g.nx), hj = min(max(y0 + hy, -1), g.ny);
        hpos = (hy + 1) * PW + hx + 1;
        hcol = (unsigned)(hi + g.gx) + (unsigned)g.sy * (unsigned)(hj + IGR_NG);
    }
    // raw loads of a plane (own column + halo cell) are issued one iteration before they are consumed
    struct Raw { float r[4], h[4]; };
    auto fetch = [&](int k, Raw &w) {
        const unsigned zo = usz * (unsigned)(min(k, g.nz) + IGR_NG);
        const unsigned o = col + zo, ho = hcol + zo;              // one 32-bit offset for the four fields
        w.r[0] = ldf(rho + o); w.r[1] = ldf(m[0] + o); w.r[2] = ldf(m[1] + o); w.r[3] = ldf(m[2] + o);
        if (hpos >= 0) {
            w.h[0] = ldf(rho + ho); w.h[1] = ldf(m[0] + ho); w.h[2] = ldf(m[1] + ho); w.h[3] = ldf(m[2] + ho);
        }
    };
    auto put_plane = [&](int buf, const Raw &w, float v[3]) {               // fetched plane -> velocities
        const float ir = __fdividef(1.0f, w.r[0]);
        v[0] = w.r[1] * ir; v[1] = w.r[2] * ir; v[2] = w.r[3] * ir;
        U[buf][0][own] = v[0]; U[buf][1][own] = v[1]; U[buf][2][own] = v[2];
        if (hpos >= 0) {
            const float hr = __fdividef(1.0f, w.h[0]);
            U[buf][0][hpos] = w.h[1] * hr; U[buf][1][hpos] = w.h[2] * hr; U[buf][2][hpos] = w.h[3] * hr;
        }
    };
    auto emit = [&](int k, const float (*P)[PN], const float dn[3], const float up[3]) {
        // without the stress fields the nine differences stay undivided: b is quadratic in them, 1/(2 dx)^2 goes
        // into the factor of the sum (nine multiplications less per cell)
        const float sc = GRAD ? inv2dx : 1.0f;
        float G[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            G[a][0] = (P[a][own + 1] - P[a][own - 1]) * sc;
            G[a][1] = (P[a][own + PW] - P[a][own - PW]) * sc;
            G[a][2] = (up[a] - dn[a]) * sc;
        }
        const float tr = G[0][0] + G[1][1] + G[2][2];
        const float trsq = G[0][0] * G[0][0] + G[1][1] * G[1][1] + G[2][2] * G[2][2] +
                           2.0f * (G[0][1] * G[1][0] + G[0][2] * G[2][0] + G[1][2] * G[2][1]);
        if (valid) {
            const unsigned id = col + usz * (unsigned)(k + IGR_NG);
            b[id] = (GRAD ? alpha : alpha * inv2dx * inv2dx) * (trsq + tr * tr);
            if (GRAD) {                       // the same second-order gradients feed the viscous stress (L232)
                const float lt = lam2 * tr, mu2 = 2.0f * mu;
                tp.t[IGR_TAU_XX][id] = mu2 * G[0][0] + lt;
                tp.t[IGR_TAU_XY][id] = mu * (G[0][1] + G[1][0]);
                tp.t[IGR_TAU_XZ][id] = mu * (G[0][2] + G[2][0]);
                tp.t[IGR_TAU_YY][id] = mu2 * G[1][1] + lt;
                tp.t[IGR_TAU_YZ][id] = mu * (G[1][2] + G[2][1]);
                tp.t[IGR_TAU_ZZ][id] = mu2 * G[2][2] + lt;
            }
        }
    };
    // own column at planes k-1, k (dn, ce) and the two planes that enter per iteration (u1, u2)
    float dn[3], ce[3], u1[3], u2[3];
    Raw A, B;
    fetch(kz0 - 1, A);
    {
        const float ir = __fdividef(1.0f, A.r[0]);
        dn[0] = A.r[1] * ir; dn[1] = A.r[2] * ir; dn[2] = A.r[3] * ir;
    }
    fetch(kz0, A);
    int bc = 0;                                              // buffer of plane k (k = kz0 + t), mod NB
    put_plane(bc, A, ce);
    // planes per barrier: two with 4-byte storage (4.94 -> 4.72 ms at 1024^3), one with 2-byte storage (two
    // measured slower there: 7.1 vs 5.2 ms)
    constexpr int PPB = (sizeof(T) == 4) ? 2 : 1;
    fetch(kz0 + 1, A);
    if (PPB == 2) fetch(kz0 + 2, B);
    constexpr int TRIP = (PPB == 2) ? 1 : 2;               // two planes per loop trip either way
#pragma unroll TRIP
    for (int t = 0; t < nkz; t += PPB) {
        const int k = kz0 + t;
        const int b1 = (bc + 1 >= NB) ? bc + 1 - NB : bc + 1, b2 = (bc + 2 >= NB) ? bc + 2 - NB : bc + 2;
        put_plane(b1, A, u1);                                // plane k + 1
        if (PPB == 2) put_plane(b2, B, u2);                  // plane k + 2 (ghost plane at the top)
        fetch(k + 1 + PPB, A);                               // land during this iteration
        if (PPB == 2) fetch(k + 2 + PPB, B);
        __syncthreads();                                     // one barrier per PPB planes
        emit(k, U[bc], dn, u1);
        if (PPB == 2) {
            if (t + 1 < nkz) emit(k + 1, U[b1], ce, u2);
#pragma unroll
            for (int a = 0; a < 3; ++a) { dn[a] = u1[a]; ce[a] = u2[a]; }
            bc = b2;
        } else {
#pragma unroll
            for (int a = 0; a < 3; ++a) { dn[a] = ce[a]; ce[a] = u1[a]; }
            bc = b1;
        }
    }
}

void launch_source(const Grid &g, int storage, StagePtrs q, float *b, float alpha, float inv2dx,
                   float *tau, float mu, float zeta, cudaStream_t st)
{
    dim3 grid((g.nx + SRC_TX - 1) / SRC_TX, (g.ny + SRC_TY - 1) / SRC_TY, (g.nz + SRC_ZC - 1) / SRC_ZC);
    TauPtrs tp;
    for (int c = 0; c < 6; ++c) tp.t[c] = tau ? tau + (size_t)c * g.np : nullptr;
    const float lam2 = zeta - 2.0f * mu / 3.0f;
    DISPATCH_STORAGE(storage, {
        if (tau) k_source<T, true><<<grid, SRC_TX * SRC_TY, 0, st>>>(g, q, b, alpha, inv2dx, tp, mu, lam2);
        else k_source<T, false><<<grid, SRC_TX * SRC_TY, 0, st>>>(g, q, b, alpha, inv2dx, tp, 0.f, 0.f);
    });
}

// ------------------------------------------------------------------------------ a3: Jacobi sweep
// Sigma/rho - alpha div(grad(Sigma)/rho) = b  (eq. 9, reading A1) on the 6-point stencil (L138),
// face density = arithmetic mean (reading A2):
//   Sigma_i <- ( b_i + k2 sum_n w_in Sigma_n ) / ( 1/rho_i + k2 sum_n w_in ),  w_in = 2/(rho_i + rho_n),
// k2 = alpha/dx^2.  Ghost values of the iterate follow the BC index map at every sweep (wrap /
// clamp), so the neighbour index is mapped instead of refreshing ghosts between sweeps; rho ghosts
// come from the filled q ghosts.
template <typename T>
__global__ void k_jacobi_sweep(Grid g, const T *__restrict__ rho, const float *__restrict__ b,
                               const T *__restrict__ sin, T *__restrict__ sout, float k2)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        const long long id = g.idx(i, j, k);
        const float rc = ldf(rho + id);
        float num = 0.f, den = 0.f;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int sgn = -1; sgn <= 1; sgn += 2) {
                int ii = i + (a == 0 ? sgn : 0), jj = j + (a == 1 ? sgn : 0), kk = k + (a == 2 ? sgn : 0);
                const float w = 2.0f / (rc + ldf(rho + g.idx(ii, jj, kk)));
                const long long ns = g.idx(map_index(ii, g.nx, g.bc[0]), map_index(jj, g.ny, g.bc[2]),
                                           map_index(kk, g.nz, g.bc[4]));
                num += w * ldf(sin + ns);
                den += w;
            }
        }
        stf(sout + id, (b[id] + k2 * num) / (1.0f / rc + k2 * den));
    }
}

void launch_jacobi_sweep(const Grid &g, int storage, const void *rho, const float *b,
                         const void *sig_in, void *sig_out, float k2, cudaStream_t st)
{
    long long n = (long long)g.nx * g.ny * g.nz;
    DISPATCH_STORAGE(storage, k_jacobi_sweep<T><<<blocks_for(n, 256), 256, 0, st>>>(
                                  g, (const T *)rho, b, (const T *)sig_in, (T *)sig_out, k2));
}

// ------------------------------------------------------------------------------ a4: RHS, simple form
// Reference-quality kernel (one thread per cell, both faces of each direction recomputed, global
// loads through L1/L2).  It defines the arithmetic the tiled kernel must reproduce:
//   reconstruction of (rho, m, E, Sigma) at the face from cells -2..3 (L132, L164, Alg. 1,
//   L205), primitives from the reconstructed conservative values (L187-L198), flux with p + Sigma
//   (eqs. 6-8), Lax-Friedrichs with lambda = max(|u_d| + c) of the two adjacent
//   cell-centred states (L132, L207-L210; reading A5), r = -sum_d (F^_{i+1/2} - F^_{i-1/2})/dx.
template <int ORDER>
__device__ __forceinline__ void reconstruct(const float f[6], float &fl, float &fr)
{
    if (ORDER == 5) {
        fl = (2.f / 60.f) * f[0] + (-13.f / 60.f) * f[1] + (47.f / 60.f) * f[2] + (27.f / 60.f) * f[3] + (-3.f / 60.f) * f[4];
        fr = (-3.f / 60.f) * f[1] + (27.f / 60.f) * f[2] + (47.f / 60.f) * f[3] + (-13.f / 60.f) * f[4] + (2.f / 60.f) * f[5];
    } else {
        fl = (-1.f / 6.f) * f[1] + (5.f / 6.f) * f[2] + (2.f / 6.f) * f[3];
        fr = (2.f / 6.f) * f[2] + (5.f / 6.f) * f[3] + (-1.f / 6.f) * f[4];
    }
}

__device__ __forceinline__ void side_flux(int d, float gm1, const float U[5], float sg, float F[5])
{
    const float ir = 1.0f / U[0];
    const float ud = U[1 + d] * ir;
    const float p = gm1 * (U[4] - 0.5f * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) * ir);
    F[0] = U[1 + d];
    F[1] = U[1] * ud; F[2] = U[2] * ud; F[3] = U[3] * ud;
    F[1 + d] += p + sg;
    F[4] = (U[4] + p + sg) * ud;
}

template <typename T>
__device__ __forceinline__ float cell_wavespeed(int d, float gamma, const StagePtrs &q, long long id)
{
    const float rho = ldf((const T *)q.f[0] + id), ir = 1.0f / rho;
    const float mx = ldf((const T *)q.f[1] + id), my = ldf((const T *)q.f[2] + id), mz = ldf((const T *)q.f[3] + id);
    const float p = (gamma - 1.0f) * (ldf((const T *)q.f[4] + id) - 0.5f * (mx * mx + my * my + mz * mz) * ir);
    const float md = d == 0 ? mx : (d == 1 ? my : mz);
    return fabsf(md * ir) + sqrtf(gamma * p * ir);
}

// numerical flux at the face between cell `id` and `id + stride` along d
template <typename T, int ORDER>
__device__ __forceinline__ void face_flux(int d, const StagePtrs &q, const T *sig, long long id,
                                          long long stride, float gamma, float F[5])
{
    float UL[5], UR[5], f[6], sl, sr;
#pragma unroll
    for (int c = 0; c < 5; ++c) {
#pragma unroll
        for (int t = 0; t < 6; ++t) f[t] = ldf((const T *)q.f[c] + id + (t - 2) * stride);
        reconstruct<ORDER>(f, UL[c], UR[c]);
    }
#pragma unroll
    for (int t = 0; t < 6; ++t) f[t] = ldf(sig + id + (t - 2) * stride);
    reconstruct<ORDER>(f, sl, sr);
    const float lam = fmaxf(cell_wavespeed<T>(d, gamma, q, id), cell_wavespeed<T>(d, gamma, q, id + stride));
    float FL[5], FR[5];
    side_flux(d, gamma - 1.0f, UL, sl, FL);
    side_flux(d, gamma - 1.0f, UR, sr, FR);
#pragma unroll
    for (int c = 0; c < 5; ++c) F[c] = 0.5f * (FL[c] + FR[c]) - 0.5f * lam * (UR[c] - UL[c]);
}

template <typename T, int ORDER>
__global__ void k_rhs_simple(Grid g, StagePtrs q, const T *__restrict__ sig, float *r0, float *r1,
                             float *r2, float *r3, float *r4, float gamma, float inv_dx)
{
    float *rr[5] = { r0, r1, r2, r3, r4 };
    const long long st[3] = { 1, g.sy, g.sz };
    const long long n = (long long)g.nx * g.ny * g.nz;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        const long long id = g.idx(i, j, k);
        float acc[5] = { 0.f, 0.f, 0.f, 0.f, 0.f };
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            // both faces go through ONE instance of the flux code (no unrolling), so that the two
            // cells sharing a face compute bitwise the same flux: exact conservation and exact
            // preservation of uniform states (P7, P8)
            float Fp[5], Fm[5];
#pragma unroll 1
            for (int side = 0; side < 2; ++side) {
                float F[5];
                face_flux<T, ORDER>(d, q, sig, side ? id - st[d] : id, st[d], gamma, F);
#pragma unroll
                for (int c = 0; c < 5; ++c) { if (side) Fm[c] = F[c]; else Fp[c] = F[c]; }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) acc[c] -= (Fp[c] - Fm[c]) * inv_dx;
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) rr[c][id] = acc[c];
    }
}

void launch_rhs_simple(const Grid &g, int storage, StagePtrs q, const void *sig, float *const r[5],
                       RhsParams p, cudaStream_t st)
{
    long long n = (long long)g.nx * g.ny * g.nz;
    unsigned int nb = blocks_for(n, 128);
    DISPATCH_STORAGE(storage, {
        if (p.order == 5)
            k_rhs_simple<T, 5><<<nb, 128, 0, st>>>(g, q, (const T *)sig, r[0], r[1], r[2], r[3], r[4], p.gamma, p.inv_dx);
        else
            k_rhs_simple<T, 3><<<nb, 128, 0, st>>>(g, q, (const T *)sig, r[0], r[1], r[2], r[3], r[4], p.gamma, p.inv_dx);
    });
}

// ------------------------------------------------------------------------------ a5/a6: update, wave speed
// SSP-RK3 of Gottlieb & Shu (L138, ref. 17 L389): every stage is a convex combination
//   q_out = a q_n + beta (q_s + dt r),  a + beta = 1,  beta = 1, 1/4, 2/3,
// evaluated as q_n + beta ((q_s - q_n) + dt r) so that r = 0, q_s = q_n returns q_n bitwise (A18).
// With `wave` the kernel also reduces max(|u_d|) + c of the NEW state (warp shuffle, then one
// atomicMax per block on the float bits, valid for non-negative floats) and flags non-finite cells.
__device__ __forceinline__ void block_reduce_wave(float v, bool bad, WaveResult *wave)
{
    __shared__ float s_max[32];
    __shared__ int s_bad;
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    bad = __any_sync(0xffffffffu, bad);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { s_max[wid] = v; if (bad) atomicOr(&s_bad, 1); }
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        v = lane < nw ? s_max[lane] : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0) {
            atomicMax(&wave->max_bits, __float_as_uint(v));
            if (s_bad) atomicOr(&wave->nonfinite, 1u);
        }
    }
}

template <typename T, bool WAVE>
__global__ void k_rk_update(Grid g, StagePtrs qn, StagePtrs qs, StagePtrs qo, const float *r0,
                            const float *r1, const float *r2, const float *r3, const float *r4,
                            float beta, float dt, float gamma, WaveResult *wave)
{
    const float *rr[5] = { r0, r1, r2, r3, r4 };
    const long long n = (long long)g.nx * g.ny * g.nz;
    float vmax = 0.f;
    bool bad = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        const long long id = g.idx(i, j, k);
        float o[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const float a = ldf((const T *)qn.f[c] + id), s = ldf((const T *)qs.f[c] + id);
            o[c] = __fmaf_rn(beta, __fmaf_rn(dt, rr[c][id], __fsub_rn(s, a)), a);
            stf((T *)qo.f[c] + id, o[c]);
            if (WAVE) o[c] = ldf((const T *)qo.f[c] + id);      // wave speed of the STORED state
        }
        if (WAVE && k >= g.wk0 && k < g.wk1)
            vmax = fmaxf(vmax, wavespeed_of(o[0], o[1], o[2], o[3], o[4], gamma, bad));
    }
    if (WAVE) block_reduce_wave(vmax, bad, wave);
}

void launch_rk_update(const Grid &g, int storage, StagePtrs qn, StagePtrs qs, StagePtrs qout,
                      float *const r[5], float beta, float dt, float gamma, WaveResult *wave,
                      cudaStream_t st)
{
    long long n = (long long)g.nx * g.ny * g.nz;
    unsigned int nb = blocks_for(n, 256, 148 * 8);
    DISPATCH_STORAGE(storage, {
        if (wave)
            k_rk_update<T, true><<<nb, 256, 0, st>>>(g, qn, qs, qout, r[0], r[1], r[2], r[3], r[4], beta, dt, gamma, wave);
        else
            k_rk_update<T, false><<<nb, 256, 0, st>>>(g, qn, qs, qout, r[0], r[1], r[2], r[3], r[4], beta, dt, gamma, wave);
    });
}

template <typename T>
__global__ void k_wavespeed(Grid g, StagePtrs q, float gamma, WaveResult *wave)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    float vmax = 0.f;
    bool bad = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        if (k < g.wk0 || k >= g.wk1) continue;
        const long long id = g.idx(i, j, k);
        vmax = fmaxf(vmax, wavespeed_of(ldf((const T *)q.f[0] + id), ldf((const T *)q.f[1] + id),
                                        ldf((const T *)q.f[2] + id), ldf((const T *)q.f[3] + id),
                                        ldf((const T *)q.f[4] + id), gamma, bad));
    }
    block_reduce_wave(vmax, bad, wave);
}

void launch_wavespeed(const Grid &g, int storage, StagePtrs q, float gamma, WaveResult *wave,
                      cudaStream_t st)
{
    long long n = (long long)g.nx * g.ny * g.nz;
    DISPATCH_STORAGE(storage, k_wavespeed<T><<<blocks_for(n, 256, 148 * 8), 256, 0, st>>>(g, q, gamma, wave));
}

// two fluids (fp32 storage): mixture wave speed, reading A21
__global__ void k_wavespeed2(Grid g, StagePtrs q, float k1, float k2, WaveResult *wave)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    float vmax = 0.f;
    bool bad = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
         t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        if (k < g.wk0 || k >= g.wk1) continue;
        const long long id = g.idx(i, j, k);
        float v[7];
#pragma unroll
        for (int c = 0; c < 7; ++c) v[c] = ((const float *)q.f[c])[id];
        vmax = fmaxf(vmax, wavespeed_of2(v, k1, k2, bad));
    }
    block_reduce_wave(vmax, bad, wave);
}

void launch_wavespeed2(const Grid &g, StagePtrs q, float k1, float k2, WaveResult *wave, cudaStream_t st)
{
    long long n = (long long)g.nx * g.ny * g.nz;
    k_wavespeed2<<<blocks_for(n, 256, 148 * 8), 256, 0, st>>>(g, q, k1, k2, wave);
}

// ------------------------------------------------------------------------------ NEXT-1: viscous fluxes
// Simple form (igr_viscous.cuh has the formulas; igr_viscous_tile.cu the streaming form): one thread per
// cell adds (H^+ - H^-)/dx of its six faces to r[1..4], both faces of a direction through one code
// instance.
template <typename T, int ORDER>
__global__ void __launch_bounds__(128) k_viscous_add(Grid g, StagePtrs q, const float *__restrict__ tau,
                                                     float *r1, float *r2, float *r3, float *r4, float inv_dx)
{
    const int i = blockIdx.x * 128 + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= g.nx) return;
    float *rr[4] = { r1, r2, r3, r4 };
    const long long st[3] = { 1, g.sy, g.sz };
    const long long id0 = g.idx(i, j, k);
    float acc[4] = { 0.f, 0.f, 0.f, 0.f };
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float Hp[4], Hm[4];
#pragma unroll 1
        for (int side = 0; side < 2; ++side) {
            const long long id = side ? id0 - st[d] : id0;          // left cell of the face
            float tq[4][6], tt[3][6], H[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
#pragma unroll
                for (int t = 0; t < 6; ++t) tq[c][t] = ldf((const T *)q.f[c] + id + (t - 2) * st[d]);
            }
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float *tf = tau + (long long)igr_visc::tau_field(d, a) * g.np;
#pragma unroll
                for (int t = 0; t < 6; ++t) tt[a][t] = tf[id + (t - 2) * st[d]];
            }
            igr_visc::face<ORDER>(tq, tt, H);
#pragma unroll
            for (int c = 0; c < 4; ++c) { if (side) Hm[c] = H[c]; else Hp[c] = H[c]; }
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[c] = __fadd_rn(acc[c], __fsub_rn(Hp[c], Hm[c]));
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) rr[c][id0] = __fmaf_rn(inv_dx, acc[c], rr[c][id0]);
}

void launch_viscous_add(const Grid &g, int storage, int order, StagePtrs q, const float *tau,
                        float *const r[5], float inv_dx, cudaStream_t st)
{
    dim3 grid((g.nx + 127) / 128, g.ny, g.nz);
    DISPATCH_STORAGE(storage, {
        if (order == 5) k_viscous_add<T, 5><<<grid, 128, 0, st>>>(g, q, tau, r[1], r[2], r[3], r[4], inv_dx);
        else k_viscous_add<T, 3><<<grid, 128, 0, st>>>(g, q, tau, r[1], r[2], r[3], r[4], inv_dx);
    });
}

// =============================================================================== fp64 mode (NEXT-4)
// IGR_STORE_F64: fp64 storage AND fp64 arithmetic, for a like-for-like column beside the paper's FP64 grind
// times (Table 1).  One thread per cell, one launch per row and per Jacobi sweep, IEEE
// division and square root, every formula in the oracle's order (parity <= 1e-12 after several steps).  It is the
// straightforward form of the hot path: the tiled TMA kernels are fp32 (the precision the paper's large runs and
// the headline use, L297); B200's plain FP64 rate is half its FP32 rate and the state is twice as large.
namespace f64 {

__global__ void k_unpack(Grid g, const double *__restrict__ user, double *__restrict__ field, int k0, int nk)
{
    long long n = (long long)nk * g.ny * g.nx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        field[g.idx(i, (int)(r % g.ny), k0 + (int)(r / g.ny))] = user[t];
    }
}
__global__ void k_unpack32(Grid g, const float *__restrict__ user, double *__restrict__ field, int k0, int nk)
{
    long long n = (long long)nk * g.ny * g.nx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        field[g.idx(i, (int)(r % g.ny), k0 + (int)(r / g.ny))] = (double)user[t];
    }
}
__global__ void k_pack(Grid g, const double *__restrict__ field, double *__restrict__ user, int k0, int nk)
{
    long long n = (long long)nk * g.ny * g.nx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        user[t] = field[g.idx(i, (int)(r % g.ny), k0 + (int)(r / g.ny))];
    }
}
__global__ void k_pack32(Grid g, const double *__restrict__ field, float *__restrict__ user, int k0, int nk)
{
    long long n = (long long)nk * g.ny * g.nx;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        user[t] = (float)field[g.idx(i, (int)(r % g.ny), k0 + (int)(r / g.ny))];
    }
}

// a1: ghosts of q by the index map, blended towards the fixed patch state on inflow faces (reading A8 / A8b)
__global__ void k_halo_q(Grid g, StagePtrs q, Inflow64 bc)
{
    const long long n = ghost_count(g);
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        GhostCell c = decode_ghost(g, t);
        if (ghost_is_external(g, c.i, c.j, c.k)) continue;
        const long long dst = g.idx(c.i, c.j, c.k);
        const long long src = g.idx(map_index(c.i, g.nx, g.bc[0]), map_index(c.j, g.ny, g.bc[2]),
                                    map_index(c.k, g.nz, g.bc[4]));
        double w = 0.0;
        const double *fixed = nullptr;
        const int idx[3] = { c.i, c.j, c.k }, nn[3] = { g.nx, g.ny, g.nz };
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int face = idx[a] < 0 ? 2 * a : (idx[a] >= nn[a] ? 2 * a + 1 : -1);
            if (face < 0 || fixed != nullptr || bc.weight[face] == nullptr) continue;
            int t0 = (a == 0) ? idx[1] : idx[0];
            int t1 = (a == 2) ? idx[1] : idx[2];
            if (t0 < 0 || t0 >= bc.n0[face] || t1 < 0 || t1 >= bc.n1[face]) continue;
            double ww = bc.weight[face][(long long)t1 * bc.n0[face] + t0];
            if (ww > 0.0) { w = ww; fixed = bc.fixed[face] + ((long long)t1 * bc.n0[face] + t0) * 5; }
        }
#pragma unroll
        for (int cmp = 0; cmp < 5; ++cmp) {
            double *fld = (double *)q.f[cmp];
            double v = fld[src];
            if (fixed != nullptr) v = (w >= 1.0) ? fixed[cmp] : v + w * (fixed[cmp] - v);
            fld[dst] = v;
        }
    }
}

__global__ void k_halo_sigma(Grid g, double *__restrict__ sig)
{
    const long long n = ghost_count(g);
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        GhostCell c = decode_ghost(g, t);
        if (ghost_is_external(g, c.i, c.j, c.k)) continue;
        sig[g.idx(c.i, c.j, c.k)] = sig[g.idx(map_index(c.i, g.nx, g.bc[0]), map_index(c.j, g.ny, g.bc[2]),
                                              map_index(c.k, g.nz, g.bc[4]))];
    }
}

// a2: b = alpha (tr((grad u)^2) + (tr grad u)^2), central differences of u = m / rho (eq. 9; L132)
__global__ void k_source(Grid g, StagePtrs q, double *__restrict__ b, double alpha, double inv2dx)
{
    const long long st[3] = { 1, g.sy, g.sz };
    const long long n = (long long)g.nx * g.ny * g.nz;
    const double *rho = (const double *)q.f[0];
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        const long long id = g.idx(i, (int)(r % g.ny), (int)(r / g.ny));
        double G[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double *m = (const double *)q.f[1 + a];
#pragma unroll
            for (int d = 0; d < 3; ++d)
                G[a][d] = (m[id + st[d]] / rho[id + st[d]] - m[id - st[d]] / rho[id - st[d]]) * inv2dx;
        }
        double trsq = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int d = 0; d < 3; ++d) trsq += G[a][d] * G[d][a];
        }
        const double tr = G[0][0] + G[1][1] + G[2][2];
        b[id] = alpha * (trsq + tr * tr);
    }
}

// a3: one Jacobi sweep; Sigma neighbours through the BC index map, densities from the filled ghosts
__global__ void k_jacobi_sweep(Grid g, const double *__restrict__ rho, const double *__restrict__ b,
                               const double *__restrict__ sin, double *__restrict__ sout, double k2)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int j = (int)(r % g.ny), k = (int)(r / g.ny);
        const long long id = g.idx(i, j, k);
        const double rc = rho[id];
        double num = 0.0, den = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
#pragma unroll
            for (int sgn = -1; sgn <= 1; sgn += 2) {
                int ii = i + (a == 0 ? sgn : 0), jj = j + (a == 1 ? sgn : 0), kk = k + (a == 2 ? sgn : 0);
                const double w = 2.0 / (rc + rho[g.idx(ii, jj, kk)]);
                num += w * sin[g.idx(map_index(ii, g.nx, g.bc[0]), map_index(jj, g.ny, g.bc[2]),
                                     map_index(kk, g.nz, g.bc[4]))];
                den += w;
            }
        }
        sout[id] = (b[id] + k2 * num) / (1.0 / rc + k2 * den);
    }
}

// a4: r = -div F^ (reconstruction L132/L164, primitives from reconstructed values L187-L198, p + Sigma eqs. 6-8,
// local Lax-Friedrichs L207-L210 with the cell-centred speed of the two adjacent cells, reading A5)
template <int ORDER>
__device__ __forceinline__ void reconstruct(const double f[6], double &fl, double &fr)
{
    if (ORDER == 5) {
        fl = (2.0 * f[0] - 13.0 * f[1] + 47.0 * f[2] + 27.0 * f[3] - 3.0 * f[4]) / 60.0;
        fr = (-3.0 * f[1] + 27.0 * f[2] + 47.0 * f[3] - 13.0 * f[4] + 2.0 * f[5]) / 60.0;
    } else {
        fl = (-f[1] + 5.0 * f[2] + 2.0 * f[3]) / 6.0;
        fr = (2.0 * f[2] + 5.0 * f[3] - f[4]) / 6.0;
    }
}

__device__ __forceinline__ void side_flux(int d, double gm1, const double U[5], double sg, double F[5])
{
    const double ud = U[1 + d] / U[0];
    const double p = gm1 * (U[4] - 0.5 * (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) / U[0]);
    F[0] = U[1 + d];
    F[1] = U[1] * ud; F[2] = U[2] * ud; F[3] = U[3] * ud;
    F[1 + d] += p + sg;
    F[4] = (U[4] + p + sg) * ud;
}

__device__ __forceinline__ double cell_wavespeed(int d, double gamma, const StagePtrs &q, long long id)
{
    const double rho = ((const double *)q.f[0])[id];
    const double mx = ((const double *)q.f[1])[id], my = ((const double *)q.f[2])[id], mz = ((const double *)q.f[3])[id];
    const double p = (gamma - 1.0) * (((const double *)q.f[4])[id] - 0.5 * (mx * mx + my * my + mz * mz) / rho);
    const double md = d == 0 ? mx : (d == 1 ? my : mz);
    return fabs(md / rho) + sqrt(gamma * p / rho);
}

template <int ORDER>
__device__ __forceinline__ void face_flux(int d, const StagePtrs &q, const double *sig, long long id, long long stride,
                                          double gamma, double F[5])
{
    double UL[5], UR[5], f[6], sl, sr;
#pragma unroll
    for (int c = 0; c < 5; ++c) {
#pragma unroll
        for (int t = 0; t < 6; ++t) f[t] = ((const double *)q.f[c])[id + (t - 2) * stride];
        reconstruct<ORDER>(f, UL[c], UR[c]);
    }
#pragma unroll
    for (int t = 0; t < 6; ++t) f[t] = sig[id + (t - 2) * stride];
    reconstruct<ORDER>(f, sl, sr);
    const double lam = fmax(cell_wavespeed(d, gamma, q, id), cell_wavespeed(d, gamma, q, id + stride));
    double FL[5], FR[5];
    side_flux(d, gamma - 1.0, UL, sl, FL);
    side_flux(d, gamma - 1.0, UR, sr, FR);
#pragma unroll
    for (int c = 0; c < 5; ++c) F[c] = 0.5 * (FL[c] + FR[c]) - 0.5 * lam * (UR[c] - UL[c]);
}

struct RPtrs { double *r[5]; };

template <int ORDER>
__global__ void __launch_bounds__(128) k_rhs(Grid g, StagePtrs q, const double *__restrict__ sig, RPtrs rr, double gamma,
                                             double dx)
{
    const long long st[3] = { 1, g.sy, g.sz };
    const long long n = (long long)g.nx * g.ny * g.nz;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        const long long id = g.idx(i, (int)(r % g.ny), (int)(r / g.ny));
        double acc[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            // both faces through ONE instance of the flux code: the two cells of a face see bitwise the same flux
            double Fp[5], Fm[5];
#pragma unroll 1
            for (int side = 0; side < 2; ++side) {
                double F[5];
                face_flux<ORDER>(d, q, sig, side ? id - st[d] : id, st[d], gamma, F);
#pragma unroll
                for (int c = 0; c < 5; ++c) { if (side) Fm[c] = F[c]; else Fp[c] = F[c]; }
            }
#pragma unroll
            for (int c = 0; c < 5; ++c) acc[c] -= (Fp[c] - Fm[c]) / dx;
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) rr.r[c][id] = acc[c];
    }
}

// a6: max_d |u_d| + c; non-negative doubles order like their bit patterns, so one 64-bit atomicMax per block
__device__ __forceinline__ void block_reduce_wave(double v, bool bad, WaveResult64 *wave)
{
    __shared__ double s_max[32];
    __shared__ int s_bad;
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    bad = __any_sync(0xffffffffu, bad);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { s_max[wid] = v; if (bad) atomicOr(&s_bad, 1); }
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        v = lane < nw ? s_max[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0) {
            atomicMax(&wave->max_bits, (unsigned long long)__double_as_longlong(v));
            if (s_bad) atomicOr(&wave->nonfinite, 1u);
        }
    }
}

__device__ __forceinline__ double wavespeed_of(const double o[5], double gamma, bool &bad)
{
    const double rho = o[0];
    const double p = (gamma - 1.0) * (o[4] - 0.5 * (o[1] * o[1] + o[2] * o[2] + o[3] * o[3]) / rho);
    const double um = fmax(fabs(o[1] / rho), fmax(fabs(o[2] / rho), fabs(o[3] / rho)));
    const double v = um + sqrt(gamma * p / rho);
    if (!(v <= 1.0e300)) { bad = true; return 0.0; }
    return v;
}

// a5 (+ a6): q_out = q_n + beta ((q_s - q_n) + dt r)  (reading A18)
template <bool WAVE>
__global__ void k_rk_update(Grid g, StagePtrs qn, StagePtrs qs, StagePtrs qo, RPtrs rr, double beta, double dt,
                            double gamma, WaveResult64 *wave)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    double vmax = 0.0;
    bool bad = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int k = (int)(r / g.ny);
        const long long id = g.idx(i, (int)(r % g.ny), k);
        double o[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double a = ((const double *)qn.f[c])[id], s = ((const double *)qs.f[c])[id];
            o[c] = a + beta * ((s - a) + dt * rr.r[c][id]);
            ((double *)qo.f[c])[id] = o[c];
        }
        if (WAVE && k >= g.wk0 && k < g.wk1) vmax = fmax(vmax, wavespeed_of(o, gamma, bad));
    }
    if (WAVE) block_reduce_wave(vmax, bad, wave);
}

__global__ void k_wavespeed(Grid g, StagePtrs q, double gamma, WaveResult64 *wave)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    double vmax = 0.0;
    bool bad = false;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        int i = (int)(t % g.nx); long long r = t / g.nx;
        int k = (int)(r / g.ny);
        if (k < g.wk0 || k >= g.wk1) continue;
        const long long id = g.idx(i, (int)(r % g.ny), k);
        double o[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) o[c] = ((const double *)q.f[c])[id];
        vmax = fmax(vmax, wavespeed_of(o, gamma, bad));
    }
    block_reduce_wave(vmax, bad, wave);
}

}  // namespace f64

// ---- fp64 launchers (igr_kernels.h)
void launch64_unpack(const Grid &g, const void *user, int user_is_f32, double *field, int k0, int nk, cudaStream_t st)
{
    const long long n = (long long)nk * g.ny * g.nx;
    if (user_is_f32) f64::k_unpack32<<<blocks_for(n, 256), 256, 0, st>>>(g, (const float *)user, field, k0, nk);
    else f64::k_unpack<<<blocks_for(n, 256), 256, 0, st>>>(g, (const double *)user, field, k0, nk);
}
void launch64_pack(const Grid &g, const double *field, void *user, int user_is_f32, int k0, int nk, cudaStream_t st)
{
    const long long n = (long long)nk * g.ny * g.nx;
    if (user_is_f32) f64::k_pack32<<<blocks_for(n, 256), 256, 0, st>>>(g, field, (float *)user, k0, nk);
    else f64::k_pack<<<blocks_for(n, 256), 256, 0, st>>>(g, field, (double *)user, k0, nk);
}
void launch64_halo_q(const Grid &g, StagePtrs q, const Inflow64 &bc, cudaStream_t st)
{
    f64::k_halo_q<<<blocks_for(ghost_count(g), 256, 148 * 16), 256, 0, st>>>(g, q, bc);
}
void launch64_halo_sigma(const Grid &g, double *sig, cudaStream_t st)
{
    f64::k_halo_sigma<<<blocks_for(ghost_count(g), 256, 148 * 16), 256, 0, st>>>(g, sig);
}
void launch64_source(const Grid &g, StagePtrs q, double *b, double alpha, double inv2dx, cudaStream_t st)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    f64::k_source<<<blocks_for(n, 256), 256, 0, st>>>(g, q, b, alpha, inv2dx);
}
void launch64_jacobi_sweep(const Grid &g, const double *rho, const double *b, const double *sin, double *sout, double k2,
                           cudaStream_t st)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    f64::k_jacobi_sweep<<<blocks_for(n, 256), 256, 0, st>>>(g, rho, b, sin, sout, k2);
}
void launch64_rhs(const Grid &g, int order, StagePtrs q, const double *sig, double *const r[5], double gamma, double dx,
                  cudaStream_t st)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    f64::RPtrs rr;
    for (int c = 0; c < 5; ++c) rr.r[c] = r[c];
    if (order == 5) f64::k_rhs<5><<<blocks_for(n, 128), 128, 0, st>>>(g, q, sig, rr, gamma, dx);
    else f64::k_rhs<3><<<blocks_for(n, 128), 128, 0, st>>>(g, q, sig, rr, gamma, dx);
}
void launch64_rk_update(const Grid &g, StagePtrs qn, StagePtrs qs, StagePtrs qout, double *const r[5], double beta,
                        double dt, double gamma, WaveResult64 *wave, cudaStream_t st)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    f64::RPtrs rr;
    for (int c = 0; c < 5; ++c) rr.r[c] = r[c];
    const unsigned nb = blocks_for(n, 256, 148 * 8);
    if (wave) f64::k_rk_update<true><<<nb, 256, 0, st>>>(g, qn, qs, qout, rr, beta, dt, gamma, wave);
    else f64::k_rk_update<false><<<nb, 256, 0, st>>>(g, qn, qs, qout, rr, beta, dt, gamma, wave);
}
void launch64_wavespeed(const Grid &g, StagePtrs q, double gamma, WaveResult64 *wave, cudaStream_t st)
{
    const long long n = (long long)g.nx * g.ny * g.nz;
    f64::k_wavespeed<<<blocks_for(n, 256, 148 * 8), 256, 0, st>>>(g, q, gamma, wave);
}
