// igr_jacobi_blocked.cu -- row a3 of the hot path for sm_100a: NS (= n_jacobi, up to 5) warm-started
// Jacobi sweeps of
//     Sigma/rho - alpha div(grad(Sigma)/rho) = b          (eq. 9; A1-A3)
// temporally blocked: ONE pass over HBM reads rho, b, Sigma_old and writes Sigma_new after all NS
// sweeps (16 B per cell instead of 16 B per sweep).
//
// Design: 2.5-D streaming with a skewed pipeline of sweep levels.
// A CTA of 512 threads (two columns per thread) owns a 32 x 32 column region = (32-2NS)^2 output columns
// + an NS-wide halo that is recomputed (the dependency cone of NS sweeps), and marches along z.  At step tau the plane
// p0 enters; level l+1 (l = 0..NS-1) advances its iterate on plane p0-1-l from level l's planes
// p0-2-l .. p0-l.  In-plane neighbours come from double-buffered shared-memory planes (one per
// level), the z neighbours and all seven stencil coefficients of the NS planes in flight live in
// registers (a compile-time rotated ring, so nothing is shifted).  One __syncthreads per plane.
// Ghost values of every iterate follow the BC index map at every sweep (wrap / clamp, reading A8):
// periodic directions are recomputed from wrapped data, clamp directions read the cell itself in
// place of its outside neighbour.
#include "igr_kernels.h"
#include "igr_tma.cuh"

#include <cuda.h>
#include <cstdlib>
#include <type_traits>

namespace {

constexpr int R = 32;                       // region edge
constexpr int cpt_small = 2;                // columns per thread for NS <= 3 (1 = 1024 threads: measured slower)

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

constexpr int PF = 3;                       // prefetch distance in planes (cp.async or TMA)
constexpr int SUB = (R + 4) * R;            // floats of one staged field: an fp32 TMA box of (R + 4) x R
// CPT = columns per thread (rows ry and ry + R/CPT of the region).  NS = 4, 5: CPT = 2, 512 threads x
// 128 registers hold the pipeline state (7 coefficients x NS planes + 2 NS iterate values per column);
// CPT = 1 (1024 threads x 64 registers, no spills for NS <= 3) was measured slower and is not used.
template <typename T, int NS, int CPT>
__global__ void __launch_bounds__(R * R / CPT, 1)
k_jacobi_blocked(const __grid_constant__ CUtensorMap rmap, const __grid_constant__ CUtensorMap bmap,
                 const __grid_constant__ CUtensorMap smap, int use_tma, Grid g, const T *__restrict__ rho,
                 const float *__restrict__ bsrc, const T *__restrict__ sin, T *__restrict__ sout, float k2, int zc,
                 JacobiQuadPlan skip)
{
    // regions taken by k_jacobi_quad (CTA-uniform)
    if ((int)blockIdx.x >= skip.bx0 && (int)blockIdx.x < skip.bx0 + skip.nbx && (int)blockIdx.y >= skip.by0 &&
        (int)blockIdx.y < skip.by0 + skip.nby_blocked)
        return;
    constexpr int OT = R - 2 * NS;
    constexpr int NTHREADS = R * R / CPT;
    constexpr int P = R + 2;                 // padded plane pitch: a border of one cell, so that the
    constexpr int PP = P * (R + 2);          // four in-plane neighbours are at constant offsets
    extern __shared__ __align__(128) float jb_smem[];
    // incoming planes are staged PF steps ahead into a ring of PF + 1 slots of (rho, b, Sigma) for the
    // R*R columns.  A region that lies inside the domain in x and y is a plain box of the padded arrays:
    // ONE thread issues three TMA loads per plane (mbarrier completion).  Regions that reach over the
    // domain boundary gather through the BC index map with one 4-byte cp.async per column and field
    // (each thread reads back only what it copied itself).
    // A TMA box must start on a 16-byte boundary of the row: it starts at the region's first column rounded
    // down to 16 bytes and is 16 bytes wider than the region; the columns sit `shift` elements into each row.
    float *STG = jb_smem;                                                               // [PF+1][3][SUB]
    float (*RHO)[PP] = reinterpret_cast<float (*)[PP]>(jb_smem + (PF + 1) * 3 * SUB);   // [2][PP]
    float (*SP)[2][PP] = reinterpret_cast<float (*)[2][PP]>(jb_smem + (PF + 1) * 3 * SUB + 2 * PP);     // [NS][2][PP]
    uint64_t *full = reinterpret_cast<uint64_t *>(jb_smem + (PF + 1) * 3 * SUB + (2 + 2 * NS) * PP);
    constexpr bool ASYNC = true;   // 2-byte storage: cp.async copies the aligned 4-byte word holding the element

    const int rx = threadIdx.x & 31, ry0 = threadIdx.x >> 5;
    const int gi = blockIdx.x * OT - NS + rx;
    const int kz0 = blockIdx.z * zc, nkz = min(zc, g.nz - kz0);
    const bool per_x = g.bc[0] == 0, per_y = g.bc[2] == 0, per_z = g.bc[4] == 0;
    const unsigned usz = (unsigned)g.sz;

    // Ghost values of every iterate follow the BC index map at every sweep.  Periodic: the halo
    // columns are wrapped real cells, recomputed.  Clamp: the ghost equals the nearest interior cell:
    // a cell on a clamp boundary also writes its value into the neighbouring ghost position, and
    // threads at positions outside a clamped domain do not store at all.
    enum { ST_OWN = 1, ST_W = 2, ST_E = 4, ST_S = 8, ST_N = 16, ST_CORE = 32 };
    int pos[CPT], mask[CPT];
    unsigned off_r[CPT], off_m[CPT], off_o[CPT];     // element offsets fit 32 bits on any grid that fits
#pragma unroll
    for (int cc = 0; cc < CPT; ++cc) {
        const int ry = ry0 + cc * (R / CPT), gj = blockIdx.y * OT - NS + ry;
        pos[cc] = (ry + 1) * P + rx + 1;
        int m = 0;
        const bool in_x = per_x || (gi >= 0 && gi < g.nx), in_y = per_y || (gj >= 0 && gj < g.ny);
        if (in_x && in_y) {
            m |= ST_OWN;
            if (!per_x && gi == 0) m |= ST_W;
            if (!per_x && gi == g.nx - 1) m |= ST_E;
            if (!per_y && gj == 0) m |= ST_S;
            if (!per_y && gj == g.ny - 1) m |= ST_N;
        }
        if (rx >= NS && rx < R - NS && ry >= NS && ry < R - NS && gi < g.nx && gj < g.ny) m |= ST_CORE;
        mask[cc] = m;
        off_r[cc] = (unsigned)(rho_index(gi, g.nx, per_x) + g.gx) +
                    (unsigned)g.sy * (unsigned)(rho_index(gj, g.ny, per_y) + IGR_NG);
        off_m[cc] = (unsigned)(map_index(gi, g.nx, g.bc[0]) + g.gx) +
                    (unsigned)g.sy * (unsigned)(map_index(gj, g.ny, g.bc[2]) + IGR_NG);
        off_o[cc] = (unsigned)(gi + g.gx) + (unsigned)g.sy * (unsigned)(gj + IGR_NG);
    }
    // CTA-uniform: does this region touch a clamp boundary of the domain in x or y (or contain
    // positions outside it)?  Interior CTAs take the variant of the loop body without any masks.
    const int gi_lo = blockIdx.x * OT - NS, gj_lo = blockIdx.y * OT - NS;
    const bool cta_edge = (!per_x && (gi_lo <= 0 || gi_lo + R >= g.nx)) || (!per_y && (gj_lo <= 0 || gj_lo + R >= g.ny));

    const bool tma_cta = use_tma && gi_lo >= 0 && gi_lo + R <= g.nx && gj_lo >= 0 && gj_lo + R <= g.ny;
    constexpr int ALT = 16 / (int)sizeof(T), BWT = R + ALT, BWB = R + 4;    // box widths: T fields / fp32 b
    const int xcol = g.gx + gi_lo, shT = xcol & (ALT - 1), shB = xcol & 3;
    auto tma_issue = [&](int p, int stage) {     // one thread: plane p of the three fields -> staging slot
        float *st = STG + stage * 3 * SUB;
        const int zr = rho_index(p, g.nz, per_z) + IGR_NG, zm = map_index(p, g.nz, g.bc[4]) + IGR_NG;
        igr_tma::mbar_expect_tx(&full[stage], R * (2 * BWT * (int)sizeof(T) + BWB * 4));
        igr_tma::tma_load_3d(st, &rmap, xcol - shT, IGR_NG + gj_lo, zr, &full[stage]);
        igr_tma::tma_load_3d(st + SUB, &bmap, xcol - shB, IGR_NG + gj_lo, zm, &full[stage]);
        igr_tma::tma_load_3d(st + 2 * SUB, &smap, xcol - shT, IGR_NG + gj_lo, zm, &full[stage]);
    };

    static_assert(PF == 3, "slot arithmetic assumes a ring of 4");
    const uint32_t full_s = igr_tma::smem_u32(full);
    unsigned slot = 0, phase = 0;            // staging slot of the plane consumed in this step, its phase

    Coef C[CPT][NS];                         // ring: coefficient set of plane p lives in slot p mod NS
    float below[CPT][NS], centre[CPT][NS];   // own column: level-l iterate at planes c-1, c (c = p1 - l)
    float rho1[CPT], b1[CPT], wz_prev[CPT], rn0[CPT], bn0[CPT], sn0[CPT];
#pragma unroll
    for (int cc = 0; cc < CPT; ++cc) {
#pragma unroll
        for (int l = 0; l < NS; ++l) {
            C[cc][l].wxm = C[cc][l].wxp = C[cc][l].wym = C[cc][l].wyp = C[cc][l].wzp = 0.f;
            C[cc][l].dinv = C[cc][l].b = 0.f;
            below[cc][l] = centre[cc][l] = 0.f;
        }
        rho1[cc] = 1.f; b1[cc] = 0.f; wz_prev[cc] = 0.f;
    }
    for (int e = threadIdx.x; e < PP; e += NTHREADS) {
        RHO[0][e] = 1.f; RHO[1][e] = 1.f;
#pragma unroll
        for (int l = 0; l < NS; ++l) { SP[l][0][e] = 0.f; SP[l][1][e] = 0.f; }
    }

    auto load_plane = [&](int p) {               // register prefetch, one step ahead (half storage)
        const unsigned zr = usz * (unsigned)(rho_index(p, g.nz, per_z) + IGR_NG);
        const unsigned zm = usz * (unsigned)(map_index(p, g.nz, g.bc[4]) + IGR_NG);
#pragma unroll
        for (int cc = 0; cc < CPT; ++cc) {
            rn0[cc] = ldf(rho + (off_r[cc] + zr));
            bn0[cc] = bsrc[off_m[cc] + zm];
            sn0[cc] = ldf(sin + (off_m[cc] + zm));
        }
    };
    auto cp4 = [](float *dst, const void *src) {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((unsigned)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
    };
    auto stage_plane = [&](int p, int stage) {   // asynchronous copy of plane p into a staging slot
        const unsigned zr = usz * (unsigned)(rho_index(p, g.nz, per_z) + IGR_NG);
        const unsigned zm = usz * (unsigned)(map_index(p, g.nz, g.bc[4]) + IGR_NG);
        float *st = STG + stage * 3 * SUB + threadIdx.x;
#pragma unroll
        for (int cc = 0; cc < CPT; ++cc) {
            // (for 2-byte T the source address is rounded down to its 4-byte word)
            constexpr uintptr_t WORD = (sizeof(T) == 4) ? ~(uintptr_t)0 : ~(uintptr_t)3;
            cp4(st + cc * NTHREADS, reinterpret_cast<const void *>(reinterpret_cast<uintptr_t>(rho + (off_r[cc] + zr)) & WORD));
            cp4(st + SUB + cc * NTHREADS, bsrc + (off_m[cc] + zm));
            cp4(st + 2 * SUB + cc * NTHREADS, reinterpret_cast<const void *>(reinterpret_cast<uintptr_t>(sin + (off_m[cc] + zm)) & WORD));
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    const int kfirst = kz0 - NS;             // first plane that enters; plane p <-> step p - kfirst
    const int nsteps = nkz + 2 * NS;         // output plane of step tau is kfirst + tau - NS
    const float k22 = 2.0f * k2;
    if (tma_cta) {
        if (threadIdx.x == 0) {
            for (int d = 0; d <= PF; ++d) igr_tma::mbar_init(&full[d], 1);
            igr_tma::fence_init();
            for (int d = 0; d < PF; ++d) tma_issue(kfirst + d, d);     // nsteps > PF always
        }
    } else if (ASYNC) {
#pragma unroll
        for (int d = 0; d < PF; ++d) stage_plane(kfirst + d, d);
    } else {
        load_plane(kfirst);
    }
    __syncthreads();

    // NS steps with compile-time ring slots; EDGE = false drops every boundary mask and select
    auto group = [&](int base, auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        auto put = [&](float *plane, int cc, float v) {
            const int ps = pos[cc];
            if (!EDGE) { plane[ps] = v; return; }
            const int m = mask[cc];
            if (m & ST_OWN) plane[ps] = v;
            if (m & ST_W) plane[ps - 1] = v;
            if (m & ST_E) plane[ps + 1] = v;
            if (m & ST_S) plane[ps - P] = v;
            if (m & ST_N) plane[ps + P] = v;
        };
#pragma unroll
        for (int u = 0; u < NS; ++u) {
            const int tau = base + u;
            const int p0 = kfirst + tau, p1 = p0 - 1;
            float rho0[CPT], b0[CPT], s0[CPT];
            if (tma_cta) {
                // the slot of plane p0 + PF was read in the previous step (barrier since): refill it
                if (threadIdx.x == 0 && tau + PF < nsteps) {
                    igr_tma::fence_async();
                    tma_issue(p0 + PF, (slot + PF) & PF);          // (slot + PF) mod (PF + 1), PF + 1 = 4
                }
                // (the last group may run a few steps past nsteps: nothing was loaded for them, their
                // values are never stored)
                if (tau < nsteps) igr_tma::mbar_wait_s32(full_s + 8u * slot, phase);
                const float *st = STG + slot * (3 * SUB);
                if (++slot == PF + 1) { slot = 0; phase ^= 1u; }
#pragma unroll
                for (int cc = 0; cc < CPT; ++cc) {
                    const int ry = ry0 + cc * (R / CPT);
                    b0[cc] = st[SUB + ry * BWB + shB + rx];
                    rho0[cc] = ldf(reinterpret_cast<const T *>(st) + (ry * BWT + shT + rx));
                    s0[cc] = ldf(reinterpret_cast<const T *>(st + 2 * SUB) + (ry * BWT + shT + rx));
                }
            } else if (ASYNC) {
                // plane p0 was committed PF steps ago; keep PF groups in flight (empty groups at the end)
                stage_plane(p0 + PF, (tau + PF) % (PF + 1));
                asm volatile("cp.async.wait_group %0;" ::"n"(PF) : "memory");
                const float *st = STG + (tau % (PF + 1)) * 3 * SUB + threadIdx.x;
#pragma unroll
                for (int cc = 0; cc < CPT; ++cc) {
                    b0[cc] = st[SUB + cc * NTHREADS];
                    if (sizeof(T) == 4) {
                        rho0[cc] = st[cc * NTHREADS]; s0[cc] = st[2 * SUB + cc * NTHREADS];
                    } else {
                        // pick the element out of its word: the parity of the element offset is the
                        // same for every plane when the plane stride is even (it is: px is a multiple of 16)
                        const T *wr = reinterpret_cast<const T *>(st + cc * NTHREADS);
                        const T *ws = reinterpret_cast<const T *>(st + 2 * SUB + cc * NTHREADS);
                        rho0[cc] = ldf(wr + (off_r[cc] & 1u)); s0[cc] = ldf(ws + (off_m[cc] & 1u));
                    }
                }
            } else {
#pragma unroll
                for (int cc = 0; cc < CPT; ++cc) { rho0[cc] = rn0[cc]; b0[cc] = bn0[cc]; s0[cc] = sn0[cc]; }
                if (tau + 1 < nsteps) load_plane(p0 + 1);                    // prefetch the next plane
            }
            const int par0 = tau & 1, par1 = par0 ^ 1;                       // parity of planes p0 / p1
            const int slot1 = (u + NS - 1) % NS;                              // ring slot of plane p1
            const int ko = p0 - NS;                                           // output plane of this step
            const bool out_ok = ko >= kz0 && ko < kz0 + nkz;
            float wz_old[CPT];
#pragma unroll
            for (int cc = 0; cc < CPT; ++cc) {
                RHO[par0][pos[cc]] = rho0[cc];
                put(SP[0][par0], cc, s0[cc]);

                // ---- coefficients of plane p1 (its densities were stored in the previous step);
                // the slot held plane p1 - NS, whose W_z+ the last level still needs
                wz_old[cc] = C[cc][slot1].wzp;
                const float *rp = &RHO[par1][pos[cc]];
                const float r1 = rho1[cc];
                Coef c;
                c.wxm = k22 * rcp_approx(r1 + rp[-1]);
                c.wxp = k22 * rcp_approx(r1 + rp[1]);
                c.wym = k22 * rcp_approx(r1 + rp[-P]);
                c.wyp = k22 * rcp_approx(r1 + rp[P]);
                c.wzp = k22 * rcp_approx(r1 + rho0[cc]);
                c.dinv = rcp_approx(rcp_approx(r1) + ((c.wxm + c.wxp) + (c.wym + c.wyp) + (wz_prev[cc] + c.wzp)));
                c.b = b1[cc];
                wz_prev[cc] = c.wzp;                                          // W_z- of the next plane
                C[cc][slot1] = c;
            }

            // ---- levels: level l+1 advances plane c = p1 - l, both columns together.  The in-plane
            // neighbours of level l+1's plane were written in the PREVIOUS step (other buffer of the
            // pair), so they are fetched one level ahead of their use, before this level's stores.
            float above[CPT], nb[CPT][4];
#pragma unroll
            for (int cc = 0; cc < CPT; ++cc) {
                above[cc] = s0[cc];                                           // level-0 iterate at plane p0
                const float *sp = &SP[0][par1][pos[cc]];
                nb[cc][0] = sp[-1]; nb[cc][1] = sp[1]; nb[cc][2] = sp[-P]; nb[cc][3] = sp[P];
            }
#pragma unroll
            for (int l = 0; l < NS; ++l) {
                const int c = p1 - l;
                const int slot = (u + 2 * NS - 1 - l) % NS;                   // slot of plane c
                const int slot_m = (u + 2 * NS - 2 - l) % NS;                 // slot of plane c - 1
                float nx[CPT][4];
                if (l + 1 < NS) {
#pragma unroll
                    for (int cc = 0; cc < CPT; ++cc) {
                        const float *sp = &SP[l + 1][(par1 + l + 1) & 1][pos[cc]];
                        nx[cc][0] = sp[-1]; nx[cc][1] = sp[1]; nx[cc][2] = sp[-P]; nx[cc][3] = sp[P];
                    }
                }
#pragma unroll
                for (int cc = 0; cc < CPT; ++cc) {
                    const Coef &k = C[cc][slot];
                    const float wzm = (l == NS - 1) ? wz_old[cc] : C[cc][slot_m].wzp;
                    const float ctr = centre[cc][l];
                    const float dn = (EDGE && !per_z && c == 0) ? ctr : below[cc][l];
                    const float up = (EDGE && !per_z && c == g.nz - 1) ? ctr : above[cc];
                    // two partial sums: shorter dependency chains
                    float a0 = fmaf(k.wxm, nb[cc][0], k.b);
                    float a1 = k.wxp * nb[cc][1];
                    a0 = fmaf(k.wym, nb[cc][2], a0);
                    a1 = fmaf(k.wyp, nb[cc][3], a1);
                    a0 = fmaf(wzm, dn, a0);
                    a1 = fmaf(k.wzp, up, a1);
                    const float fresh = (a0 + a1) * k.dinv;                   // level l+1 at plane c
                    below[cc][l] = ctr;
                    centre[cc][l] = above[cc];
                    above[cc] = fresh;
                    if (l + 1 < NS) put(SP[l + 1][(par1 + l) & 1], cc, fresh);
                }
                if (l + 1 < NS) {
#pragma unroll
                    for (int cc = 0; cc < CPT; ++cc) {
#pragma unroll
                        for (int n = 0; n < 4; ++n) nb[cc][n] = nx[cc][n];
                    }
                }
            }
#pragma unroll
            for (int cc = 0; cc < CPT; ++cc) {
                // above[] now holds the level-NS iterate at plane p1 - (NS - 1) = p0 - NS
                if ((mask[cc] & ST_CORE) && out_ok) stf(sout + (off_o[cc] + usz * (unsigned)(ko + IGR_NG)), above[cc]);
                rho1[cc] = rho0[cc]; b1[cc] = b0[cc];
            }
            __syncthreads();
        }
    };
    for (int base = 0; base < nsteps; base += NS) {
        // planes touched by the levels of this group: kfirst + base - NS .. kfirst + base + NS - 1
        const int plo = kfirst + base - NS, phi = kfirst + base + NS;
        const bool z_edge = !per_z && ((plo <= 0 && phi >= 0) || (plo <= g.nz - 1 && phi >= g.nz - 1));
        if (cta_edge || z_edge) group(base, std::true_type());
        else group(base, std::false_type());
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

namespace {

// 3-D map (x, y, z) of one padded field; box = region + 16 bytes in x (the box start is rounded down to 16 B)
bool encode_plane_map(CUtensorMap *out, const Grid &g, const void *base, int storage, int rows)
{
    const size_t es = storage == 0 ? 4 : 2;
    cuuint64_t dims[3] = { (cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz };
    cuuint64_t strides[2] = { (cuuint64_t)g.px * es, (cuuint64_t)g.px * g.py * es };
    cuuint32_t box[3] = { (cuuint32_t)(R + 16 / es), (cuuint32_t)rows, 1 };     // 16 bytes wider than the region
    return igr_tma::encode(out, igr_tma::data_type(storage), 3, base, dims, strides, box);
}

}  // namespace

int jacobi_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state, void *const sig[2],
                     const float *b, JacobiMaps *out, int rows)
{
    out->valid = false;
    for (int i = 0; i < 3; ++i)
        if (!encode_plane_map(&out->rho[i], g, st[i < n_state ? i : n_state - 1].f[0], storage, rows)) return 1;
    for (int i = 0; i < 2; ++i)
        if (!encode_plane_map(&out->sig[i], g, sig[i], storage, rows)) return 1;
    if (!encode_plane_map(&out->b, g, b, 0, rows)) return 1;
    out->valid = true;
    return 0;
}

template <typename T>
static void launch_ns(const Grid &g, int ns, const void *rho, const float *b, const void *sin, void *sout,
                      float k2, const CUtensorMap *rmap, const CUtensorMap *bmap, const CUtensorMap *smap,
                      const JacobiQuadPlan &skip, cudaStream_t st)
{
    const int ot = R - 2 * ns, zc = jacobi_blocked_zc(g, ns);
    dim3 grid((g.nx + ot - 1) / ot, (g.ny + ot - 1) / ot, (g.nz + zc - 1) / zc);
    const int use_tma = (rmap && bmap && smap) ? 1 : 0;
    static const CUtensorMap dummy = {};
    const CUtensorMap &rm = use_tma ? *rmap : dummy, &bm = use_tma ? *bmap : dummy, &sm = use_tma ? *smap : dummy;
#define IGR_JB_SMEM(NSV) ((2 + 2 * (NSV)) * (R + 2) * (R + 2) * 4 + (PF + 1) * 3 * SUB * 4 + (PF + 1) * 8 + 8)
    const int smem = IGR_JB_SMEM(ns);
#define IGR_JB(NSV)                                                                                      \
    do {                                                                                                 \
        constexpr int CPTV = (NSV <= 3) ? cpt_small : 2;                                                 \
        static bool configured = false;                                                                  \
        if (!configured) {                                                                               \
            cudaFuncSetAttribute(k_jacobi_blocked<T, NSV, CPTV>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                 IGR_JB_SMEM(NSV));                                                      \
            configured = true;                                                                           \
        }                                                                                                \
        k_jacobi_blocked<T, NSV, CPTV><<<grid, R * R / CPTV, smem, st>>>(rm, bm, sm, use_tma, g, (const T *)rho, b, \
                                                                    (const T *)sin, (T *)sout, k2, zc, skip);  \
    } while (0)
    switch (ns) {
    case 1: IGR_JB(1); break;
    case 2: IGR_JB(2); break;
    case 3: IGR_JB(3); break;
    case 4: IGR_JB(4); break;
    default: IGR_JB(5); break;
    }
#undef IGR_JB
#undef IGR_JB_SMEM
}

// ns in 1..5 sweeps in one pass; sig_in and sig_out must differ.  With the three maps (planes of rho, b and
// sig_in) regions inside the domain stage their planes by TMA; NULL maps: cp.async everywhere.
void launch_jacobi_blocked(const Grid &g, int storage, int ns, const void *rho, const float *b,
                           const void *sig_in, void *sig_out, float k2, const CUtensorMap *rmap,
                           const CUtensorMap *bmap, const CUtensorMap *smap, const JacobiQuadPlan *skip,
                           cudaStream_t st)
{
    JacobiQuadPlan none = {};
    const JacobiQuadPlan &sk = skip ? *skip : none;
    if (sk.nbx > 0 && sk.nby > 0) {
        // every region is taken by the quad kernel: nothing to launch
        const int ot = R - 2 * ns;
        if (sk.bx0 == 0 && sk.by0 == 0 && sk.nbx >= (g.nx + ot - 1) / ot && sk.nby_blocked >= (g.ny + ot - 1) / ot) return;
    }
    if (storage == 0) launch_ns<float>(g, ns, rho, b, sig_in, sig_out, k2, rmap, bmap, smap, sk, st);
    else if (storage == 1) launch_ns<__half>(g, ns, rho, b, sig_in, sig_out, k2, rmap, bmap, smap, sk, st);
    else launch_ns<__nv_bfloat16>(g, ns, rho, b, sig_in, sig_out, k2, rmap, bmap, smap, sk, st);
}
