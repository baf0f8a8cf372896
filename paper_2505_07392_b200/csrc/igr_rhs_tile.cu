// igr_rhs_tile.cu -- row a4 of the hot path for sm_100a: r = -div F^ from (q, Sigma), optionally fused
// with the RK stage update (a5) and the wave-speed reduction (a6).
//
// Design: 2.5-D streaming.  A CTA owns a 32 x TY column of cells and marches
// along z.  Whole xy-planes of the six fields (q[5] as one 4-D box, Sigma as a 3-D box) with their
// 3-cell halos are staged into a 7-slot shared-memory ring by TMA (cp.async.bulk.tensor + mbarrier),
// three planes ahead of use.  Each thread owns one (x, y) column: the z stencil lives in a sliding
// register window (6 planes x 6 fields), the x and y stencils are read from the current plane in
// shared memory.  Every face flux is computed exactly once per CTA: a thread computes the right (x+),
// top (y+) and upper (z+) face of its cell; the x- face comes from the neighbouring lane by shuffle,
// the y- face through shared memory, the z- face from the previous plane step (registers).  The
// faces on the tile's low x and y edges are computed by two designated warps.  No atomics: each cell
// differences its own six faces (gather form), so sums are deterministic and both cells adjacent to a
// face see bitwise the same flux (conservation to round-off, uniform states preserved exactly).
//
// Arithmetic (same as k_rhs_simple): Alg. 1, eqs. 6-8 L119-L125.
#include "igr_rhs_tile.cuh"
#include "igr_tma.cuh"

#include <cstdio>
#include <cstdlib>
#include <cuda_fp16.h>
#include <cuda_bf16.h>

namespace {

constexpr int TX = 32;          // tile width = warp width
#ifndef IGR_RHS_NSLOT2
#define IGR_RHS_NSLOT2 6        // ring slots of the two-fluid kernel (8 fields per plane)
#endif

using namespace igr_tma;

__device__ __forceinline__ float rcp_fast(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float sqrt_fast(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- geometry of one ring slot for storage type T
// NF = conserved fields (5: single fluid; 7: two fluids, reading A21)
template <typename T, int TY, int NF = 5, int NSLOT_OF_T = (NF == 5 ? 7 : IGR_RHS_NSLOT2)>
struct Tile {
    static constexpr int NC = NF == 5 ? 5 : NF + 1;      // flux components exchanged per face (two fluids: + u^)
    static constexpr int NSLOT = NSLOT_OF_T;             // ring slots (planes): 4 live + 2 or 3 in flight
    static constexpr int HX = 16 / (int)sizeof(T);       // x halo of the box: 4 (fp32) / 8 (half) -> 16 B
    static constexpr int BX = TX + 2 * HX;               // box extents
    static constexpr int BY = TY + 6;
    static constexpr int PE = BX * BY;                   // elements of one field in a plane
    static constexpr int QBYTES = (NF * PE * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int SBYTES = (PE * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int SLOT = QBYTES + SBYTES;          // bytes per slot
    static constexpr int TXBYTES = (NF + 1) * PE * (int)sizeof(T); // bytes one plane's two TMA loads deliver
    static constexpr int AW = TX + 2;                     // width of the wave-speed arrays (halo 1)
    static constexpr int RING = NSLOT * SLOT;
    // everything below is double-buffered by plane / step parity: one __syncthreads per plane
    static constexpr int A_N = (TY + 2) * AW;                        // floats of one wave-speed array
    static constexpr int A_OFF = RING;                               // float [2][ax | ay][A_N]
    static constexpr int FY_OFF = A_OFF + 2 * 2 * A_N * 4;           // float [2][NC][TY][TX]
    static constexpr int EX_OFF = FY_OFF + 2 * NC * TY * TX * 4;     // float [2][NC][TY]
    static constexpr int EY_OFF = EX_OFF + 2 * NC * TY * 4;          // float [2][NC][TX]
    static constexpr int BAR_OFF = (EY_OFF + 2 * NC * TX * 4 + 7) / 8 * 8;
    static constexpr int TOTAL = BAR_OFF + NSLOT * 8;
};

template <typename T> __device__ __forceinline__ float lds(const T *p);
template <> __device__ __forceinline__ float lds<float>(const float *p) { return *p; }
template <> __device__ __forceinline__ float lds<__half>(const __half *p) { return __half2float(*p); }
template <> __device__ __forceinline__ float lds<__nv_bfloat16>(const __nv_bfloat16 *p) { return __bfloat162float(*p); }

// ---- numerical flux at one face from the six stencil cells of the six fields.
// t[p][s]: field pair p (struct Pairs), stencil cell s = 0..5 <-> cells -2..3 about the face.
// Returns G = 2 F^ = (F_L + F_R) - lambda (U_R - U_L); the factor 1/2 is folded into the divergence.
// Written with explicit round-to-nearest intrinsics (never contracted or re-associated), so that every
// inlined instance -- main path, edge warps, neighbouring CTAs -- produces bitwise the same flux from
// the same inputs (conservation to round-off; uniform states preserved exactly, P7/P8).
// Packed arithmetic (sm_100: FFMA2 / FADD2 / FMUL2, two fp32 operations per issue slot, each rounded exactly like the
// scalar instruction).  The fields and the flux components travel in PAIRS: one packed instruction serves two fields.
// The kernel is bound by instruction issue, so this is where the time goes; the pairs are chosen so that no
// value ever has to be moved between register pairs.
typedef float2 f2;
__device__ __forceinline__ f2 splat(float c) { return make_float2(c, c); }
__device__ __forceinline__ f2 fsub2(f2 a, f2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }   // FADD2 a, -b

// NF = 5: (m_x, m_y), (m_z, E), (rho, Sigma);  NF = 7: (a1 rho1, a2 rho2), (m_x, m_y), (m_z, E), (a1, Sigma).
// Flux components sit where their field sits; the face velocity u^ of two fluids takes Sigma's place.
template <int NF>
struct Pairs {
    static constexpr int NP = (NF + 1) / 2;
    __host__ __device__ static constexpr int fa(int p) { return NF == 5 ? (p == 2 ? 0 : 2 * p + 1) : 2 * p; }
    __host__ __device__ static constexpr int fb(int p) { return NF == 5 ? (p == 2 ? 5 : 2 * p + 2) : 2 * p + 1; }
    __host__ __device__ static constexpr int pr(int f) { return NF == 5 ? ((f == 0 || f == 5) ? 2 : (f - 1) / 2) : f / 2; }
    __host__ __device__ static constexpr int hf(int f) { return NF == 5 ? (f == 0 ? 0 : f == 5 ? 1 : (f - 1) % 2) : f % 2; }
};
template <int NF>
__device__ __forceinline__ float pget(const f2 *v, int f)
{
    return Pairs<NF>::hf(f) ? v[Pairs<NF>::pr(f)].y : v[Pairs<NF>::pr(f)].x;
}
template <int NF>
__device__ __forceinline__ void pset(f2 *v, int f, float x)
{
    if (Pairs<NF>::hf(f)) v[Pairs<NF>::pr(f)].y = x; else v[Pairs<NF>::pr(f)].x = x;
}

template <int ORDER>
__device__ __forceinline__ void recon(const f2 t[6], f2 &l, f2 &r)
{
    if (ORDER == 5) {
        l = __fmul2_rn(splat(2.f / 60.f), t[0]);
        l = __ffma2_rn(splat(-13.f / 60.f), t[1], l);
        l = __ffma2_rn(splat(47.f / 60.f), t[2], l);
        l = __ffma2_rn(splat(27.f / 60.f), t[3], l);
        l = __ffma2_rn(splat(-3.f / 60.f), t[4], l);
        r = __fmul2_rn(splat(-3.f / 60.f), t[1]);
        r = __ffma2_rn(splat(27.f / 60.f), t[2], r);
        r = __ffma2_rn(splat(47.f / 60.f), t[3], r);
        r = __ffma2_rn(splat(-13.f / 60.f), t[4], r);
        r = __ffma2_rn(splat(2.f / 60.f), t[5], r);
    } else {
        l = __fmul2_rn(splat(-1.f / 6.f), t[1]);
        l = __ffma2_rn(splat(5.f / 6.f), t[2], l);
        l = __ffma2_rn(splat(2.f / 6.f), t[3], l);
        r = __fmul2_rn(splat(2.f / 6.f), t[2]);
        r = __ffma2_rn(splat(5.f / 6.f), t[3], r);
        r = __ffma2_rn(splat(-1.f / 6.f), t[4], r);
    }
}

// Equation of state handed to the flux routines.  Single fluid: p = (gamma - 1) e.  Two fluids (reading A21): the
// isobaric mixture rule p = e / Gamma, Gamma = a1/(gamma_1 - 1) + (1 - a1)/(gamma_2 - 1) = a1 (k1 - k2) + k2.
struct Eos {
    float gamma, gm1;      // single fluid
    float k1, k2;          // two fluids: 1/(gamma_i - 1)
};

// physical flux of one side along D from the reconstructed conservative values U[0..NF-1] and Sigma U[NF].
// NF = 5: U = (rho, m, E), F = (m_d, m u_d + (p + Sigma) e_d, (E + p + Sigma) u_d)              (eqs. 6-8).
// NF = 7: U = (a1 rho1, a2 rho2, m, E, a1), F = (a1 rho1 u_d, a2 rho2 u_d, ..., a1 u_d), and F[7] = u_d (for u^).
template <int D, int NF>
__device__ __forceinline__ void side_flux2(const float *U, const Eos &eos, float *F)
{
    constexpr int IM = NF == 5 ? 1 : 2, IE = IM + 3;
    const float rho = NF == 5 ? U[0] : __fadd_rn(U[0], U[1]);
    const float ir = rcp_fast(rho);
    const float ud = __fmul_rn(U[IM + D], ir);
    float m2 = __fmul_rn(U[IM], U[IM]);
    m2 = __fmaf_rn(U[IM + 1], U[IM + 1], m2);
    m2 = __fmaf_rn(U[IM + 2], U[IM + 2], m2);
    const float e = __fmaf_rn(__fmul_rn(-0.5f, ir), m2, U[IE]);    // E - |m|^2/(2 rho)
    float pt;                                                      // p + Sigma
    if (NF == 5) {
        pt = __fmaf_rn(eos.gm1, e, U[NF]);
        F[0] = U[IM + D];
    } else {
        const float g1 = rcp_fast(__fmaf_rn(U[6], eos.k1 - eos.k2, eos.k2));   // 1 / Gamma(a1)
        pt = __fmaf_rn(g1, e, U[NF]);
        F[0] = __fmul_rn(U[0], ud);
        F[1] = __fmul_rn(U[1], ud);
        F[6] = __fmul_rn(U[6], ud);
        F[7] = ud;
    }
    F[IM] = (D == 0) ? __fmaf_rn(U[IM], ud, pt) : __fmul_rn(U[IM], ud);
    F[IM + 1] = (D == 1) ? __fmaf_rn(U[IM + 1], ud, pt) : __fmul_rn(U[IM + 1], ud);
    F[IM + 2] = (D == 2) ? __fmaf_rn(U[IM + 2], ud, pt) : __fmul_rn(U[IM + 2], ud);
    F[IE] = __fmul_rn(__fadd_rn(U[IE], pt), ud);
}

// G = 2 F^ for the NF conserved fields, in pairs (G[p] holds the components of the fields of pair p); two fluids:
// the second half of the last pair is u_d,L + u_d,R = 2 u^ (the face velocity of a1 div u)
template <int ORDER, int D, int NF>
__device__ __forceinline__ void face_flux2(const f2 t[][6], float lam, const Eos &eos, f2 *G)
{
    using PM = Pairs<NF>;
    constexpr int NC = NF == 5 ? 5 : NF + 1;
    f2 L2[PM::NP], R2[PM::NP];
#pragma unroll
    for (int p = 0; p < PM::NP; ++p) recon<ORDER>(t[p], L2[p], R2[p]);
    float L[NF + 1], R[NF + 1];
#pragma unroll
    for (int f = 0; f < NF + 1; ++f) { L[f] = pget<NF>(L2, f); R[f] = pget<NF>(R2, f); }
    float FL[NC], FR[NC];
    side_flux2<D, NF>(L, eos, FL);
    side_flux2<D, NF>(R, eos, FR);
#pragma unroll
    for (int p = 0; p < PM::NP; ++p) {
        if (NF == 5 && p == 2) {          // rho alone (Sigma has no flux)
            G[p].x = __fmaf_rn(-lam, __fsub_rn(R[0], L[0]), __fadd_rn(FL[0], FR[0]));
            G[p].y = 0.f;
        } else {
            const f2 fl = make_float2(FL[PM::fa(p)], FL[PM::fb(p)]), fr = make_float2(FR[PM::fa(p)], FR[PM::fb(p)]);
            // (u^ carries no dissipation: its multiplier is zero)
            const f2 nl = make_float2(-lam, (NF != 5 && p == PM::NP - 1) ? 0.f : -lam);
            G[p] = __ffma2_rn(nl, fsub2(R2[p], L2[p]), __fadd2_rn(fl, fr));
        }
    }
}

// cell-centred wave speeds |u_d| + c of one cell (reading A5); explicit intrinsics as above.
// q[0..NF-1]: the conserved values of the cell.  c^2 = gamma p / rho, two fluids: (1 + 1/Gamma) p / rho.
template <int NF>
__device__ __forceinline__ void cell_speeds(const float *q, const Eos &eos, float &ax, float &ay, float &az)
{
    constexpr int IM = NF == 5 ? 1 : 2, IE = IM + 3;
    const float rho = NF == 5 ? q[0] : __fadd_rn(q[0], q[1]);
    const float ir = rcp_fast(rho);
    float m2 = __fmul_rn(q[IM], q[IM]);
    m2 = __fmaf_rn(q[IM + 1], q[IM + 1], m2);
    m2 = __fmaf_rn(q[IM + 2], q[IM + 2], m2);
    const float e = __fmaf_rn(__fmul_rn(-0.5f, ir), m2, q[IE]);
    float gg;                                                      // gamma (gamma - 1), or (1 + 1/Gamma)/Gamma
    if (NF == 5) gg = __fmul_rn(eos.gamma, eos.gm1);
    else {
        const float g1 = rcp_fast(__fmaf_rn(q[6], eos.k1 - eos.k2, eos.k2));
        gg = __fmul_rn(__fadd_rn(1.0f, g1), g1);
    }
    const float c = sqrt_fast(__fmul_rn(gg, __fmul_rn(e, ir)));
    ax = __fadd_rn(fabsf(__fmul_rn(q[IM], ir)), c);
    ay = __fadd_rn(fabsf(__fmul_rn(q[IM + 1], ir)), c);
    az = __fadd_rn(fabsf(__fmul_rn(q[IM + 2], ir)), c);
}

}  // namespace

// ======================================================================================= kernel
template <typename T, int TY, int ORDER, bool FUSE, int NF>
__global__ void __launch_bounds__(TX * TY, (TY <= 8 && NF == 5) ? 2 : 1)
k_rhs_tile(const __grid_constant__ CUtensorMap qmap, const __grid_constant__ CUtensorMap smap, Grid g,
           RhsTileArgs a)
{
    using TL = Tile<T, TY, NF>;
    constexpr int NC = TL::NC;                                          // flux components per face
    using PM = Pairs<NF>;
    constexpr int NP = PM::NP;                                          // pairs of fields in the window: q and Sigma
    constexpr bool TWO = NF != 5;
    extern __shared__ __align__(1024) unsigned char smem[];
    float *Abase = reinterpret_cast<float *>(smem + TL::A_OFF);         // [2][ax | ay][(TY+2)][AW]
    float *FYbase = reinterpret_cast<float *>(smem + TL::FY_OFF);       // [2][NC][TY][TX]
    float *EXbase = reinterpret_cast<float *>(smem + TL::EX_OFF);       // [2][NC][TY]
    float *EYbase = reinterpret_cast<float *>(smem + TL::EY_OFF);       // [2][NC][TX]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + TL::BAR_OFF);

    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5, warp = ty;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int kz0 = blockIdx.z * a.zc;
    const int nkz = min(a.zc, g.nz - kz0);
    const int i = x0 + tx, j = y0 + ty;
    const bool valid = (i < g.nx) && (j < g.ny);
    Eos eos;
    eos.gamma = a.gamma; eos.gm1 = a.gamma - 1.0f; eos.k1 = a.k1; eos.k2 = a.k2;
    const float hdx = 0.5f * a.inv_dx;                 // G = 2 F^

    // TMA coordinates of the box origin in the padded arrays (elements)
    const int cx = g.gx + x0 - TL::HX, cy = y0, cz0 = kz0;       // plane p <-> padded z = kz0 + p
    auto issue = [&](int p, int slot) {                           // one elected thread; slot = p mod TL::NSLOT
        unsigned char *dst = smem + slot * TL::SLOT;
        mbar_expect_tx(&full[slot], TL::TXBYTES);
        tma_load_4d(dst, &qmap, cx, cy, cz0 + p, 0, &full[slot]);
        tma_load_3d(dst + TL::QBYTES, &smap, cx, cy, cz0 + p, &full[slot]);
    };
    const int n_planes = nkz + 6;                                  // planes kz0-3 .. kz0+nkz+2
    if (tid == 0) {
        for (int s = 0; s < TL::NSLOT; ++s) mbar_init(&full[s], 1);
        fence_init();
        for (int p = 0; p < TL::NSLOT; ++p) issue(p, p);               // n_planes >= 7 >= TL::NSLOT
    }
    __syncthreads();

    const int own = (3 + ty) * TL::BX + TL::HX + tx;               // own cell inside a plane box
    // slot = plane index mod TL::NSLOT; the march keeps the slot indices as wrapping counters (no division)
    auto qbase = [&](int slot) { return reinterpret_cast<const T *>(smem + slot * TL::SLOT); };
    auto sbase = [&](int slot) { return reinterpret_cast<const T *>(smem + slot * TL::SLOT + TL::QBYTES); };

    // ---- prologue: window of planes p = 0..5 (cells kz0-3 .. kz0+2), flux of the face kz0-1/2
    f2 W[NP][6];                                                   // W[p][s]: pair p of the fields (struct Pairs)
#pragma unroll
    for (int s = 0; s < 6; ++s) {
        mbar_wait(&full[s], 0);
        const T *qb = qbase(s) + own, *sb = sbase(s) + own;
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            W[p][s].x = lds<T>(PM::fa(p) < NF ? qb + PM::fa(p) * TL::PE : sb);
            W[p][s].y = lds<T>(PM::fb(p) < NF ? qb + PM::fb(p) * TL::PE : sb);
        }
    }
    // the conserved values of the own column at window position s
    auto column = [&](int s, float *q) {
#pragma unroll
        for (int f = 0; f < NF; ++f) q[f] = PM::hf(f) ? W[PM::pr(f)][s].y : W[PM::pr(f)][s].x;
    };
    f2 Gz_prev[NP];
    float ax_c, ay_c, az_c;
    {
        float bx, by, az_m, q2[NF], q3[NF];
        column(2, q2); column(3, q3);
        cell_speeds<NF>(q2, eos, bx, by, az_m);                    // cell kz0-1
        cell_speeds<NF>(q3, eos, ax_c, ay_c, az_c);                // cell kz0
        face_flux2<ORDER, 2, NF>(W, fmaxf(az_m, az_c), eos, Gz_prev);
        (void)bx; (void)by;
    }
#pragma unroll
    for (int p = 0; p < NP; ++p) {
#pragma unroll
        for (int s = 0; s < 5; ++s) W[p][s] = W[p][s + 1];          // now cells kz0-2 .. kz0+2 in W[.][0..4]
    }
    // cell-centred wave speeds |u_d| + c of plane p (own cells from registers, the halo ring of the
    // tile from the ring slot) into the buffer of that plane's parity
    auto put_speeds = [&](int p, int slot, float oax, float oay) {
        float *A0 = Abase + (p & 1) * 2 * TL::A_N, *A1 = A0 + TL::A_N;
        A0[(ty + 1) * TL::AW + tx + 1] = oax;
        A1[(ty + 1) * TL::AW + tx + 1] = oay;
        // (warps 4, 5, 6 take 32 halo cells each: warps 2 and 3 have the edge faces, and the step ends at a barrier)
        if (warp >= 4 && warp < 7) {
            // x-halo (tx = -1, 32) needs ax, y-halo (ty = -1, TY) needs ay
            const T *qp = qbase(slot);
            const int h = (warp - 4) * 32 + tx;
            if (h < 2 * TY + 2 * TX) {
                int hx, hy;
                if (h < 2 * TY) { hx = (h & 1) ? TX : -1; hy = h >> 1; }
                else { const int hh = h - 2 * TY; hy = (hh >= TX) ? TY : -1; hx = hh & (TX - 1); }
                const T *c0 = qp + (3 + hy) * TL::BX + TL::HX + hx;
                float hq[NF], hax, hay, haz;
#pragma unroll
                for (int f = 0; f < NF; ++f) hq[f] = lds<T>(c0 + f * TL::PE);
                cell_speeds<NF>(hq, eos, hax, hay, haz);
                A0[(hy + 1) * TL::AW + hx + 1] = hax;
                A1[(hy + 1) * TL::AW + hx + 1] = hay;
            }
        }
    };
    put_speeds(3, 3, ax_c, ay_c);                                  // plane of the first cell layer kz0
    __syncthreads();                                               // planes 0..2 are no longer needed
    if (tid == 0) {
        fence_async();
        for (int p = TL::NSLOT; p < TL::NSLOT + 3 && p < n_planes; ++p) issue(p, p - TL::NSLOT);
    }

    float vmax = 0.f;
    bool bad = false;
    // element offsets fit 32 bits (unsigned) on any grid that fits the device
    unsigned uid = (unsigned)(min(i, g.nx - 1) + g.gx) + (unsigned)g.sy * (unsigned)(min(j, g.ny - 1) + IGR_NG) +
                   (unsigned)g.sz * (unsigned)(kz0 + IGR_NG);

    // ---- march: step t computes cell plane k = kz0 + t; current plane p = t + 3
    int slot_c = 3, slot_n = 6 % TL::NSLOT, phase_n = (6 / TL::NSLOT) & 1;  // slots of planes t + 3 and t + 6
    // two plane steps per loop trip: half of the register-window moves become renames and the parity of the
    // double-buffered exchange arrays is a compile-time constant (25.1 -> 23.7 ms; 3 and 4 steps per trip: 26.3 / 27.7 ms)
#pragma unroll 2
    for (int t = 0; t < nkz; ++t) {
        const int pc = t + 3;
        const int slot_c1 = (slot_c == TL::NSLOT - 1) ? 0 : slot_c + 1;  // slot of plane pc + 1
        mbar_wait(&full[slot_n], phase_n);
        {
            const T *qb = qbase(slot_n) + own, *sb = sbase(slot_n) + own;
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                W[p][5].x = lds<T>(PM::fa(p) < NF ? qb + PM::fa(p) * TL::PE : sb);
                W[p][5].y = lds<T>(PM::fb(p) < NF ? qb + PM::fb(p) * TL::PE : sb);
            }
        }
        // fused update: q^n of this cell is fetched now and consumed at the end of the step, so that
        // the global-load latency hides behind the flux computation
        f2 qn_pre[NP];
        const unsigned id = uid;                                    // element offset of cell (i, j, kz0 + t)
        uid += (unsigned)g.sz;
        if (FUSE && a.read_qn) {                                   // (columns beyond the domain read a valid
#pragma unroll                                                      //  cell: the offset is clamped, nothing is stored)
            for (int c = 0; c < NF; ++c) pset<NF>(qn_pre, c, ldf(reinterpret_cast<const T *>(a.qn[c]) + id));
        }
        // wave speeds of the next cell (k+1) of this column, published for the next step
        float ax_n, ay_n, az_n;
        {
            float q3[NF];
            column(3, q3);
            cell_speeds<NF>(q3, eos, ax_n, ay_n, az_n);
        }
        put_speeds(pc + 1, slot_c1, ax_n, ay_n);                  // read in the next step (after the barrier)
        // the current plane as seen by the stencil taps: the ring slot itself (2-byte storage: every tap is
        // converted where it is read -- 66 conversions per cell, but no second pass through shared memory)
        typedef T TC;
        const TC *qc = qbase(slot_c);
        const float *A0 = Abase + (pc & 1) * 2 * TL::A_N, *A1 = A0 + TL::A_N;
        float *FY = FYbase + (t & 1) * NC * TY * TX, *EX = EXbase + (t & 1) * NC * TY, *EY = EYbase + (t & 1) * NC * TX;

        const TC *sc = sbase(slot_c);
        // the six taps of every field pair about a face: `at` = the box position of stencil cell 0, `st` = the tap stride
        auto taps = [&](f2 tp[][6], int at, int st, bool own_col) {
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                const TC *pa = (PM::fa(p) < NF ? qc + PM::fa(p) * TL::PE : sc) + at;
                const TC *pb = (PM::fb(p) < NF ? qc + PM::fb(p) * TL::PE : sc) + at;
#pragma unroll
                for (int s = 0; s < 6; ++s) {
                    if (own_col && s == 2) tp[p][s] = W[p][2];          // the own cell is in the window
                    else { tp[p][s].x = lds<TC>(pa + s * st); tp[p][s].y = lds<TC>(pb + s * st); }
                }
            }
        };
        f2 Gx[NP], Gy[NP];
        {   // x+ face of the own cell: cells i-2 .. i+3
            f2 tp[NP][6];
            taps(tp, own - 2, 1, true);
            face_flux2<ORDER, 0, NF>(tp, fmaxf(ax_c, A0[(ty + 1) * TL::AW + tx + 2]), eos, Gx);
        }
        {   // y+ face: cells j-2 .. j+3
            f2 tp[NP][6];
            taps(tp, own - 2 * TL::BX, TL::BX, true);
            face_flux2<ORDER, 1, NF>(tp, fmaxf(ay_c, A1[(ty + 2) * TL::AW + tx + 1]), eos, Gy);
#pragma unroll
            for (int c = 0; c < NC; ++c) FY[(c * TY + ty) * TX + tx] = pget<NF>(Gy, c);
        }
        if (warp == 2 % TY && tx < TY) {
            // faces on the tile's low-x edge: between box columns HX-1 | HX of row tx
            f2 tp[NP][6], Ge[NP];
            taps(tp, (3 + tx) * TL::BX + TL::HX - 3, 1, false);
            face_flux2<ORDER, 0, NF>(tp, fmaxf(A0[(tx + 1) * TL::AW + 0], A0[(tx + 1) * TL::AW + 1]), eos, Ge);
#pragma unroll
            for (int c = 0; c < NC; ++c) EX[c * TY + tx] = pget<NF>(Ge, c);
        }
        if (warp == 3 % TY) {
            // faces on the tile's low-y edge: between box rows 2 | 3 of column tx
            f2 tp[NP][6], Ge[NP];
            taps(tp, TL::HX + tx, TL::BX, false);
            face_flux2<ORDER, 1, NF>(tp, fmaxf(A1[0 * TL::AW + tx + 1], A1[1 * TL::AW + tx + 1]), eos, Ge);
#pragma unroll
            for (int c = 0; c < NC; ++c) EY[c * TX + tx] = pget<NF>(Ge, c);
        }
        __syncthreads();                                   // the only barrier of the step
        if (tid == 0 && t + 3 + TL::NSLOT < n_planes) {              // slot of plane pc is free again
            fence_async();
            issue(t + 3 + TL::NSLOT, slot_c);
        }

        // z+ face (cells k-2 .. k+3 of the own column), then the divergence
        f2 Gz[NP];
        face_flux2<ORDER, 2, NF>(W, fmaxf(az_c, az_n), eos, Gz);
        f2 r[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const int ca = PM::fa(p), cb = PM::fb(p);              // components of this pair (cb may be none)
            f2 gxm, gym;
            gxm.x = __shfl_up_sync(0xffffffffu, Gx[p].x, 1);
            if (tx == 0) gxm.x = EX[ca * TY + ty];
            gym.x = (ty == 0) ? EY[ca * TX + tx] : FY[(ca * TY + ty - 1) * TX + tx];
            // r = -(1/dx) sum_d (F^+ - F^-) with G = 2 F^
            if (cb < NC) {
                gxm.y = __shfl_up_sync(0xffffffffu, Gx[p].y, 1);
                if (tx == 0) gxm.y = EX[cb * TY + ty];
                gym.y = (ty == 0) ? EY[cb * TX + tx] : FY[(cb * TY + ty - 1) * TX + tx];
                f2 acc = fsub2(Gx[p], gxm);
                acc = __fadd2_rn(acc, fsub2(Gy[p], gym));
                acc = __fadd2_rn(acc, fsub2(Gz[p], Gz_prev[p]));
                r[p] = __fmul2_rn(splat(-hdx), acc);
            } else {
                float acc = __fsub_rn(Gx[p].x, gxm.x);
                acc = __fadd_rn(acc, __fsub_rn(Gy[p].x, gym.x));
                acc = __fadd_rn(acc, __fsub_rn(Gz[p].x, Gz_prev[p].x));
                r[p].x = __fmul_rn(-hdx, acc);
                r[p].y = 0.f;
            }
            Gz_prev[p] = Gz[p];
        }
        // two fluids: + a1 div u with the face velocities u^ (the last pair holds r of a1 and -(1/dx) sum_d (u^+ - u^-))
        if (TWO) r[NP - 1].x = __fmaf_rn(-W[NP - 1][2].x, r[NP - 1].y, r[NP - 1].x);
        if (valid) {
            if (!FUSE) {
#pragma unroll
                for (int c = 0; c < NF; ++c) a.r[c][id] = pget<NF>(r, c);
            } else {
                f2 o2[NP];
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    const f2 qs = W[p][2];
                    if (PM::fb(p) < NF) {
                        const f2 qn = a.read_qn ? qn_pre[p] : qs;
                        o2[p] = __ffma2_rn(splat(a.beta), __ffma2_rn(splat(a.dt), r[p], fsub2(qs, qn)), qn);
                    } else {                                       // (x, Sigma): one field
                        const float qn = a.read_qn ? qn_pre[p].x : qs.x;
                        o2[p].x = __fmaf_rn(a.beta, __fmaf_rn(a.dt, r[p].x, __fsub_rn(qs.x, qn)), qn);
                        o2[p].y = 0.f;
                    }
                }
                float o[NF];
#pragma unroll
                for (int c = 0; c < NF; ++c) {
                    o[c] = pget<NF>(o2, c);
                    stf(reinterpret_cast<T *>(a.qout[c]) + id, o[c]);
                }
                if (a.wave && kz0 + t >= g.wk0 && kz0 + t < g.wk1) {
                    if (sizeof(T) < 4) {
#pragma unroll
                        for (int c = 0; c < NF; ++c) o[c] = ldf(reinterpret_cast<const T *>(a.qout[c]) + id);
                    }
                    if (TWO) vmax = fmaxf(vmax, wavespeed_of2(o, eos.k1, eos.k2, bad));
                    else vmax = fmaxf(vmax, wavespeed_of(o[0], o[1], o[2], o[3], o[4], a.gamma, bad));
                }
            }
        }
        // slide the window
#pragma unroll
        for (int p = 0; p < NP; ++p) {
#pragma unroll
            for (int s = 0; s < 5; ++s) W[p][s] = W[p][s + 1];
        }
        ax_c = ax_n; ay_c = ay_n; az_c = az_n;
        slot_c = slot_c1;
        if (++slot_n == TL::NSLOT) { slot_n = 0; phase_n ^= 1; }
    }

    if (FUSE && a.wave) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
        const bool anybad = __any_sync(0xffffffffu, bad);
        if (tx == 0) {
            atomicMax(&a.wave->max_bits, __float_as_uint(vmax));
            if (anybad) atomicOr(&a.wave->nonfinite, 1u);
        }
    }
}

// ======================================================================================= host
namespace {

// two fluids: 168 registers per thread, one CTA per SM: 12 rows (384 threads) fill the register file
#ifndef IGR_RHS_TY2
#define IGR_RHS_TY2 12
#endif
constexpr int TY2 = IGR_RHS_TY2;

int tile_ty(const Grid &g)
{
    static int force = -1;                       // IGR_RHS_TY=8|16 overrides the heuristic (tuning)
    if (force < 0) { const char *e = getenv("IGR_RHS_TY"); force = e ? atoi(e) : 0; }
    if (force == 8 || force == 16) return force;
    return 8;   // 2 CTAs of 256 threads per SM hide the per-plane barriers better than one of 512 (measured)
}

}  // namespace

int rhs_tile_default_zc(const Grid &g)
{
    // enough CTAs for ~4 waves of 148 SMs x (1 or 2) CTAs, chunks of at least 32 planes
    const int ty = tile_ty(g);
    const long long cols = (long long)((g.nx + TX - 1) / TX) * ((g.ny + ty - 1) / ty);
    const long long want = 4LL * 148 * (ty == 8 ? 2 : 1);
    long long nch = (want + cols - 1) / cols;
    if (nch < 1) nch = 1;
    int zc = (int)((g.nz + nch - 1) / nch);
    if (zc < 32) zc = 32;
    if (zc > g.nz) zc = g.nz;
    return zc;
}

int rhs_tile_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state, void *const sig[2],
                       int nf, RhsTileMaps *out, const char **err)
{
    out->valid = false;
    if (!igr_tma::get_encode()) { *err = "cuTensorMapEncodeTiled entry point not available"; return 1; }
    const size_t es = storage == 0 ? 4 : 2;
    const CUtensorMapDataType dt = igr_tma::data_type(storage);
    const int hx = 16 / (int)es, ty = nf == 7 ? TY2 : tile_ty(g);
    const cuuint32_t bx = TX + 2 * hx, by = ty + 6;
    for (int b = 0; b < 3; ++b) {
        const StagePtrs &s = st[b < n_state ? b : n_state - 1];
        const cuuint64_t fstride = (cuuint64_t)((char *)s.f[1] - (char *)s.f[0]);
        cuuint64_t dims[4] = { (cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz, (cuuint64_t)nf };
        cuuint64_t strides[3] = { (cuuint64_t)g.px * es, (cuuint64_t)g.px * g.py * es, fstride };
        cuuint32_t box[4] = { bx, by, 1, (cuuint32_t)nf };
        if (!igr_tma::encode(&out->q[b], dt, 4, s.f[0], dims, strides, box)) { *err = "cuTensorMapEncodeTiled(q) failed"; return 2; }
    }
    for (int b = 0; b < 2; ++b) {
        cuuint64_t dims[3] = { (cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz };
        cuuint64_t strides[2] = { (cuuint64_t)g.px * es, (cuuint64_t)g.px * g.py * es };
        cuuint32_t box[3] = { bx, by, 1 };
        if (!igr_tma::encode(&out->sig[b], dt, 3, sig[b], dims, strides, box)) { *err = "cuTensorMapEncodeTiled(sigma) failed"; return 2; }
    }
    out->valid = true;
    return 0;
}

namespace {

template <typename T, int TY, int ORDER, bool FUSE, int NF = 5>
void launch_one(const Grid &g, const CUtensorMap &qmap, const CUtensorMap &smap, RhsTileArgs a, cudaStream_t st)
{
    using TL = Tile<T, TY, NF>;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_rhs_tile<T, TY, ORDER, FUSE, NF>, cudaFuncAttributeMaxDynamicSharedMemorySize, TL::TOTAL);
        configured = true;
    }
    dim3 grid((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + a.zc - 1) / a.zc);
    k_rhs_tile<T, TY, ORDER, FUSE, NF><<<grid, TX * TY, TL::TOTAL, st>>>(qmap, smap, g, a);
}

template <typename T>
void launch_t(const Grid &g, int order, bool fused, const CUtensorMap &qmap, const CUtensorMap &smap,
              RhsTileArgs a, cudaStream_t st)
{
    const int ty = tile_ty(g);
#define IGR_CASE(TYV, ORD, FU) launch_one<T, TYV, ORD, FU>(g, qmap, smap, a, st)
    if (ty == 16) {
        if (order == 5) { if (fused) IGR_CASE(16, 5, true); else IGR_CASE(16, 5, false); }
        else { if (fused) IGR_CASE(16, 3, true); else IGR_CASE(16, 3, false); }
    } else {
        if (order == 5) { if (fused) IGR_CASE(8, 5, true); else IGR_CASE(8, 5, false); }
        else { if (fused) IGR_CASE(8, 3, true); else IGR_CASE(8, 3, false); }
    }
#undef IGR_CASE
}

}  // namespace

void launch_rhs_tile(const Grid &g, int storage, int order, bool fused, const CUtensorMap &qmap,
                     const CUtensorMap &smap, RhsTileArgs a, cudaStream_t st)
{
    if (a.zc <= 0) a.zc = rhs_tile_default_zc(g);
    if (a.nf == 7) {
        // two fluids (NEXT-3): fp32 storage, order 5, 32 x 8 tiles (igr_create_ex refuses the other combinations)
        if (fused) launch_one<float, TY2, 5, true, 7>(g, qmap, smap, a, st);
        else launch_one<float, TY2, 5, false, 7>(g, qmap, smap, a, st);
        return;
    }
    if (storage == 0) launch_t<float>(g, order, fused, qmap, smap, a, st);
    else if (storage == 1) launch_t<__half>(g, order, fused, qmap, smap, a, st);
    else launch_t<__nv_bfloat16>(g, order, fused, qmap, smap, a, st);
}
