// igr_jacobi_quad.cu -- row a3 of the hot path for sm_100a, fast path: the NS = n_jacobi warm-started Jacobi
// sweeps of
//     Sigma/rho - alpha div(grad(Sigma)/rho) = b          (eq. 9; A1-A3)
// temporally blocked in ONE pass over HBM, for every column region that needs no periodic wrap in x or y
// (igr_jacobi_blocked.cu keeps the regions that reach over a periodic boundary: it gathers through the index map).
//
// Why a second kernel: the ncu profile of k_jacobi_blocked showed the shared-memory
// data pipe as the limiter (44 four-byte words per column and plane through LDS/STS at 1 wavefront/clk/SM,
// 68 % busy; SHFL shares that pipe, measured).  Here a thread owns FOUR y-adjacent columns (lanes along x, a warp
// owns 4 rows of the 32 x 32 region, 8 warps):
//   * y neighbours inside the quad are registers; only the two edge rows of a quad go through shared memory
//     (2 STS + 2 LDS per level instead of 4 STS + 16 LDS);
//   * x neighbours come from the adjacent lane by shuffle, and only ONE x face weight per cell is kept: the
//     lane that owns the face forms W * Sigma and shuffles the product;
//   * the level-0 iterate and the densities are never re-published: neighbours read the TMA-staged planes;
//   * 20 words per column and plane instead of 44, 13 instead of 28 reciprocals per quad, and no address or
//     mask arithmetic at all (regions are plain boxes: three TMA loads per plane issued by one thread).
// The pipeline is the one of k_jacobi_blocked: 2.5-D streaming along z with a skewed pipeline of sweep
// levels; at step tau the plane p0 enters and level l+1 advances plane p0-1-l.  The z neighbours and all
// coefficients of the NS planes in flight live in registers (compile-time rotated ring).
#include "igr_kernels.h"
#include "igr_tma.cuh"

#include <cuda.h>
#include <cstdlib>
#include <type_traits>

namespace {

constexpr int R = 32;                       // region edge = warp width
constexpr int PF = 3;                       // planes in flight (TMA)
constexpr int NSLOT = PF + 2;               // + the plane that enters and the one before (its halo rows are still read)
constexpr int SBW = 12;                     // CTAs are ordered in strips of SBW regions: one wave of 148 is compact

__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// QR = rows per thread (4: 8 warps x 255 registers; 2: 16 warps x 128 registers).
// WY: the staged boxes hold the row above and the row below the 32 thread rows as well (34 rows).  Those two rows only
// ever provide the level-0 iterate and the density, which come from the staged planes anyway, so the dependency cone
// starts one row further out and 24 rows of a region are output instead of 22, at no cost (used when every y region is
// taken by this kernel, i.e. y is not periodic: the regions then need not line up with those of k_jacobi_blocked).
template <typename T, int NS, int QR, bool WY>
__global__ void __launch_bounds__(R * (R / QR), 1)
k_jacobi_quad(const __grid_constant__ CUtensorMap rmap, const __grid_constant__ CUtensorMap bmap,
              const __grid_constant__ CUtensorMap smap, Grid g, T *__restrict__ sout, float k2, int zc,
              int bx0, int by0, int nbx, int nby)
{
    constexpr int OT = R - 2 * NS, OTY = WY ? OT + 2 : OT, HY = WY ? NS - 1 : NS;   // outputs per region, y halo rows
    constexpr int ROWS = WY ? R + 2 : R, R0 = WY ? 1 : 0;  // staged rows, staged row of thread row 0
    constexpr int SUB = ((R + 4) * ROWS + 31) / 32 * 32;   // floats of one staged field (128-byte multiple: TMA)
    constexpr int NW = R / QR;                             // warps per CTA
    constexpr int NL = NS > 1 ? NS - 1 : 1;                // levels whose edge rows are exchanged
    extern __shared__ __align__(128) float jq_smem[];
    float *STG = jq_smem;                                                       // [NSLOT][3][SUB]
    float *EP = jq_smem + NSLOT * 3 * SUB;                                      // [NL][2][NW][2][32]
    uint64_t *full = reinterpret_cast<uint64_t *>(EP + NL * 2 * NW * 2 * 32);   // [NSLOT]

    // ---- which region: strips of SBW regions in x, y inside a strip, z chunks outermost
    int bx, by, bz;
    {
        const int nreg = nbx * nby;
        bz = blockIdx.x / nreg;
        const int rid = blockIdx.x - bz * nreg;
        const int nfull = nbx / SBW, wl = nbx - nfull * SBW;
        if (rid < nfull * SBW * nby) {
            const int s = rid / (SBW * nby), rem = rid - s * (SBW * nby);
            by = rem / SBW; bx = s * SBW + (rem - by * SBW);
        } else {
            const int rem = rid - nfull * SBW * nby;
            by = rem / wl; bx = nfull * SBW + (rem - by * wl);
        }
        bx += bx0; by += by0;
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, row0 = w * QR;
    const int gi_lo = bx * OT - NS, gj_lo = by * OTY - HY;         // first thread column / row of the region
    const int kz0 = bz * zc, nkz = min(zc, g.nz - kz0);
    const bool per_z = g.bc[4] == 0;
    const unsigned usz = (unsigned)g.sz;

    // ---- staging geometry (same boxes as k_jacobi_blocked): the box starts at the region's first column
    // rounded down to 16 bytes; the columns sit `sh` elements into each row
    constexpr int ALT = 16 / (int)sizeof(T), BWT = R + ALT, BWB = R + 4;
    const int xcol = g.gx + gi_lo, shT = xcol & (ALT - 1), shB = xcol & 3;
    const int own_t = (row0 + R0) * BWT + shT + lane, own_b = (row0 + R0) * BWB + shB + lane;
    // row above / below the quad (without WY the own row at the region edge: outside the dependency cone)
    const int up_t = (WY ? row0 : max(row0 - 1, 0)) * BWT + shT + lane;
    const int dn_t = (WY ? row0 + QR + 1 : min(row0 + QR, R - 1)) * BWT + shT + lane;
    // one elected lane of warp 0: plane p of the three fields -> a staging slot.  Everything it needs is
    // warp-uniform (uniform registers, no broadcast loops): the z index of the plane is a running counter kept
    // by all threads (periodic z: wrapped; otherwise rho keeps the first ghost layer, whose density enters the
    // face weights, and b, Sigma follow the index map).
    const int wu = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    auto elect_one = []() {
        uint32_t pred;
        asm volatile("{\n .reg .pred P;\n elect.sync _|P, 0xffffffff;\n selp.u32 %0, 1, 0, P;\n}" : "=r"(pred));
        return pred != 0;
    };
    auto tma_issue = [&](int p, int pwrap, int stage) {
        float *st = STG + stage * 3 * SUB;
        const int zr = (per_z ? pwrap : min(max(p, -1), g.nz)) + IGR_NG;
        const int zm = (per_z ? pwrap : min(max(p, 0), g.nz - 1)) + IGR_NG;
        igr_tma::mbar_expect_tx(&full[stage], ROWS * (2 * BWT * (int)sizeof(T) + BWB * 4));
        igr_tma::tma_load_3d(st, &rmap, xcol - shT, IGR_NG + gj_lo - R0, zr, &full[stage]);
        igr_tma::tma_load_3d(st + SUB, &bmap, xcol - shB, IGR_NG + gj_lo - R0, zm, &full[stage]);
        igr_tma::tma_load_3d(st + 2 * SUB, &smap, xcol - shT, IGR_NG + gj_lo - R0, zm, &full[stage]);
    };

    // edge rows of the quads, levels 1 .. NS-1, double-buffered by plane parity: [par][l - 1][warp][top | bottom][32].
    // Per-thread bases (row above: the bottom row of the warp above; own rows at the region edge, which is
    // outside the dependency cone); levels are compile-time offsets.
    constexpr int LSTR = NW * 2 * 32, PSTR = NL * LSTR;
    const float *const e_up = EP + ((w > 0 ? w - 1 : 0) * 2 + (w > 0 ? 1 : 0)) * 32 + lane;
    const float *const e_dn = EP + ((w < NW - 1 ? w + 1 : w) * 2 + (w < NW - 1 ? 0 : 1)) * 32 + lane;
    float *const e_own = EP + (w * 2) * 32 + lane;

    // output: core columns of the region that lie inside the domain (bit r of cmask: row r of the quad)
    unsigned cmask = 0;
#pragma unroll
    for (int r = 0; r < QR; ++r) {
        const int ry = row0 + r;
        if (lane >= NS && lane < R - NS && ry >= HY && ry < R - HY && gi_lo + lane < g.nx && gj_lo + ry < g.ny)
            cmask |= 1u << r;
    }
    // element (gi, gj of row 0, plane kz0) of the output; rows are g.sy apart, planes g.sz
    T *outp = sout + ((size_t)(gi_lo + lane + g.gx) + (size_t)g.sy * (size_t)(gj_lo + row0 + IGR_NG) +
                      (size_t)g.sz * (size_t)(kz0 + IGR_NG));
    const unsigned usy = (unsigned)g.sy;

    // Clamp boundaries in x / y (reading A8: the ghost of every iterate equals the nearest interior cell): a cell
    // on the boundary reads ITSELF in place of its outside neighbour; the face weight still comes from the real
    // ghost density (inflow ghosts differ from the clamp value).  Positions outside the domain compute garbage
    // that no valid cell reads (TMA fills rows outside the padded array with zeros).
    const int gi = gi_lo + lane;
    const bool cta_edge = gi_lo < 0 || gi_lo + R > g.nx || gj_lo < 0 || gj_lo + R > g.ny;
    const bool is_w = gi == 0, is_e = gi == g.nx - 1;
    bool is_s[QR], is_n[QR];
#pragma unroll
    for (int r = 0; r < QR; ++r) {
        const int gj = gj_lo + row0 + r;
        is_s[r] = gj == 0; is_n[r] = gj == g.ny - 1;
    }

    // ---- pipeline state.  Coefficient ring: the set of plane p lives in slot p mod NS.
    float wxp[QR][NS], wy[QR + 1][NS], wzp[QR][NS], dinv[QR][NS], bb[QR][NS];
    float below[QR][NS], centre[QR][NS];     // own columns: level-l iterate at planes c-1, c (c = p1 - l)
    float rho1[QR], b1[QR], wz_prev[QR];
#pragma unroll
    for (int r = 0; r < QR; ++r) {
#pragma unroll
        for (int l = 0; l < NS; ++l) {
            wxp[r][l] = wzp[r][l] = dinv[r][l] = bb[r][l] = 0.f;
            below[r][l] = centre[r][l] = 0.f;
        }
        rho1[r] = 1.f; b1[r] = 0.f; wz_prev[r] = 0.f;
    }
#pragma unroll
    for (int r = 0; r <= QR; ++r) {
#pragma unroll
        for (int l = 0; l < NS; ++l) wy[r][l] = 0.f;
    }
    for (int e = threadIdx.x; e < NL * 2 * NW * 2 * 32; e += R * NW) EP[e] = 0.f;

    const int kfirst = kz0 - NS;             // first plane that enters; plane p <-> step p - kfirst
    const int nsteps = nkz + 2 * NS;         // output plane of step tau is kfirst + tau - NS
    // The update is evaluated with numerator and denominator divided by 2 alpha/dx^2 =: K (plan: K is in a safe
    // range): Sigma_i = (b_i/K + sum_n W_in Sigma_n) / (1/(K rho_i) + sum_n W_in), W_in = 1/(rho_i + rho_n).
    const float k22 = 2.0f * k2, ik22 = 1.0f / k22;
    const int nsteps_r = (nsteps + NS - 1) / NS * NS;       // whole groups: the surplus steps load valid planes
    int zwrap = kfirst % g.nz;               // wrapped index of the next plane to issue (periodic z)
    if (zwrap < 0) zwrap += g.nz;
    if (threadIdx.x == 0) {
        for (int d = 0; d < NSLOT; ++d) igr_tma::mbar_init(&full[d], 1);
        igr_tma::fence_init();
    }
    __syncthreads();
    for (int d = 0; d < PF; ++d) {                                     // nsteps > PF always
        if (wu == 0 && elect_one()) tma_issue(kfirst + d, zwrap, d);
        if (++zwrap == g.nz) zwrap = 0;
    }

    const uint32_t full_s = igr_tma::smem_u32(full);
    unsigned slot = 0, phase = 0;            // staging slot of plane p0
    const float *st1 = STG;                  // staged plane p1 (step 0: no p1 yet, any finite plane will do)
    int gpar = 0;                            // parity of the first plane p1 of the group

    // NS steps with compile-time ring slots; ZEDGE: one of the planes touched is a clamp boundary in z;
    // EDGE: the region touches a clamp boundary in x / y
    auto group = [&](int base, auto zedge_tag, auto edge_tag) {
        constexpr bool ZEDGE = decltype(zedge_tag)::value, EDGE = decltype(edge_tag)::value;
        // edge-row buffers by parity relative to the group: set A holds (plane parity == gpar)
        const int oa = gpar * PSTR, ob = PSTR - oa;
#pragma unroll
        for (int u = 0; u < NS; ++u) {
            const int tau = base + u;
            const int p0 = kfirst + tau, p1 = p0 - 1;
            // the slot of plane p0 + PF held plane p0 - 2, last read in the previous step (barrier since)
            if (wu == 0 && tau + PF < nsteps_r) {
                unsigned fs = slot + PF; if (fs >= NSLOT) fs -= NSLOT;
                if (elect_one()) {
                    igr_tma::fence_async();
                    tma_issue(p0 + PF, zwrap, fs);
                }
            }
            if (++zwrap == g.nz) zwrap = 0;
            igr_tma::mbar_wait_s32(full_s + 8u * slot, phase);
            const float *st0 = STG + slot * (3 * SUB);
            if (++slot == NSLOT) { slot = 0; phase ^= 1u; }

            float rho0[QR], b0[QR], above[QR];
#pragma unroll
            for (int r = 0; r < QR; ++r) {
                rho0[r] = ldf(reinterpret_cast<const T *>(st0) + (own_t + r * BWT));
                b0[r] = st0[SUB + own_b + r * BWB];
                above[r] = ldf(reinterpret_cast<const T *>(st0 + 2 * SUB) + (own_t + r * BWT));   // level 0 at plane p0
            }
            const int slot1 = (u + NS - 1) % NS;                              // ring slot of plane p1
            const int ko = p0 - NS;                                           // output plane of this step

            // ---- coefficients of plane p1 (its own densities are registers, the rows above / below the
            // quad are still staged); the slot held plane p1 - NS, whose W_z+ the last level still needs
            float wz_old[QR];
            {
                const float r_up = ldf(reinterpret_cast<const T *>(st1) + up_t);
                const float r_dn = ldf(reinterpret_cast<const T *>(st1) + dn_t);
#pragma unroll
                for (int r = 0; r < QR; ++r) {
                    wz_old[r] = wzp[r][slot1];
                    const float r_xp = __shfl_down_sync(0xffffffffu, rho1[r], 1);
                    wxp[r][slot1] = rcp_approx(rho1[r] + r_xp);
                    wzp[r][slot1] = rcp_approx(rho1[r] + rho0[r]);
                }
                wy[0][slot1] = rcp_approx(rho1[0] + r_up);
#pragma unroll
                for (int r = 1; r < QR; ++r) wy[r][slot1] = rcp_approx(rho1[r - 1] + rho1[r]);
                wy[QR][slot1] = rcp_approx(rho1[QR - 1] + r_dn);
#pragma unroll
                for (int r = 0; r < QR; ++r) {
                    const float wxm = __shfl_up_sync(0xffffffffu, wxp[r][slot1], 1);
                    dinv[r][slot1] = rcp_approx(rcp_approx(k22 * rho1[r]) + ((wxm + wxp[r][slot1]) +
                                                                             (wy[r][slot1] + wy[r + 1][slot1]) +
                                                                             (wz_prev[r] + wzp[r][slot1])));
                    bb[r][slot1] = b1[r];
                    wz_prev[r] = wzp[r][slot1];                               // W_z- of the next plane
                }
            }

            // ---- levels: level l+1 advances plane c = p1 - l.  In-plane neighbours of level l at plane c:
            // x from the adjacent lanes (their registers), y inside the quad from registers, the rows above /
            // below the quad from the staged plane (l = 0) or from the edge rows published in the previous step.
#pragma unroll
            for (int l = 0; l < NS; ++l) {
                const int c = p1 - l;
                const int sc = (u + 2 * NS - 1 - l) % NS;                     // slot of plane c
                const int sm = (u + 2 * NS - 2 - l) % NS;                     // slot of plane c - 1
                const int eo = ((u + l) & 1) ? ob : oa;                       // buffers of plane parity (p1 + l) & 1
                float y_up, y_dn;
                if (l == 0) {
                    y_up = ldf(reinterpret_cast<const T *>(st1 + 2 * SUB) + up_t);
                    y_dn = ldf(reinterpret_cast<const T *>(st1 + 2 * SUB) + dn_t);
                } else {
                    y_up = e_up[eo + (l - 1) * LSTR];
                    y_dn = e_dn[eo + (l - 1) * LSTR];
                }
                float fresh[QR];
#pragma unroll
                for (int r = 0; r < QR; ++r) {
                    const float ctr = centre[r][l];
                    float x_p = __shfl_down_sync(0xffffffffu, ctr, 1);
                    float pm = __shfl_up_sync(0xffffffffu, wxp[r][sc] * ctr, 1);         // W_x- Sigma_x-1
                    float ym = r == 0 ? y_up : centre[r - 1][l];
                    float yp = r == QR - 1 ? y_dn : centre[r + 1][l];
                    if (EDGE) {
                        const float wxm = __shfl_up_sync(0xffffffffu, wxp[r][sc], 1);
                        if (is_w) pm = wxm * ctr;
                        if (is_e) x_p = ctr;
                        if (is_s[r]) ym = ctr;
                        if (is_n[r]) yp = ctr;
                    }
                    const float wzm = (l == NS - 1) ? wz_old[r] : wzp[r][sm];
                    const float dn = (ZEDGE && !per_z && c == 0) ? ctr : below[r][l];
                    const float up = (ZEDGE && !per_z && c == g.nz - 1) ? ctr : above[r];
                    float a = bb[r][sc] + pm;
                    a = fmaf(wxp[r][sc], x_p, a);
                    a = fmaf(wy[r][sc], ym, a);
                    a = fmaf(wy[r + 1][sc], yp, a);
                    a = fmaf(wzm, dn, a);
                    a = fmaf(wzp[r][sc], up, a);
                    fresh[r] = a * dinv[r][sc];                               // level l+1 at plane c
                }
#pragma unroll
                for (int r = 0; r < QR; ++r) {
                    below[r][l] = centre[r][l];
                    centre[r][l] = above[r];
                    above[r] = fresh[r];
                }
                if (l + 1 < NS) {
                    e_own[eo + l * LSTR] = fresh[0];
                    e_own[eo + l * LSTR + 32] = fresh[QR - 1];
                }
            }
            // above[] now holds the level-NS iterate at plane p1 - (NS - 1) = p0 - NS
            if ((unsigned)(ko - kz0) < (unsigned)nkz) {
#pragma unroll
                for (int r = 0; r < QR; ++r)
                    if (cmask & (1u << r)) stf(outp + r * usy, above[r]);
                outp += usz;
            }
#pragma unroll
            for (int r = 0; r < QR; ++r) { rho1[r] = rho0[r]; b1[r] = b0[r] * ik22; }
            st1 = st0;
            __syncthreads();
        }
        if (NS & 1) gpar ^= 1;
    };
    for (int base = 0; base < nsteps_r; base += NS) {
        // planes touched by the levels of this group: kfirst + base - NS .. kfirst + base + NS - 1
        const int plo = kfirst + base - NS, phi = kfirst + base + NS;
        const bool z_edge = !per_z && ((plo <= 0 && phi >= 0) || (plo <= g.nz - 1 && phi >= g.nz - 1));
        if (cta_edge) {
            if (z_edge) group(base, std::true_type(), std::true_type());
            else group(base, std::false_type(), std::true_type());
        } else {
            if (z_edge) group(base, std::true_type(), std::false_type());
            else group(base, std::false_type(), std::false_type());
        }
    }
}

template <typename T, int NS, int QR, bool WY>
void launch_quad(const Grid &g, const JacobiQuadPlan &pl, void *sout, float k2, const CUtensorMap &rm,
                 const CUtensorMap &bm, const CUtensorMap &sm, cudaStream_t st)
{
    constexpr int NL = NS > 1 ? NS - 1 : 1, NW = R / QR, ROWS = WY ? R + 2 : R, SUB = ((R + 4) * ROWS + 31) / 32 * 32;
    constexpr int smem = (NSLOT * 3 * SUB + NL * 2 * NW * 2 * 32) * 4 + NSLOT * 8 + 8;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_jacobi_quad<T, NS, QR, WY>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        configured = true;
    }
    const int nch = (g.nz + pl.zc - 1) / pl.zc;
    k_jacobi_quad<T, NS, QR, WY><<<pl.nbx * pl.nby * nch, R * NW, smem, st>>>(rm, bm, sm, g, (T *)sout, k2, pl.zc, pl.bx0,
                                                                      pl.by0, pl.nbx, pl.nby);
}

}  // namespace

// Regions (bx, by) of edge 32 with origin (bx OT - ns, by OT - ns), OT = 32 - 2 ns, that this kernel takes:
// bx0 <= bx < bx0 + nbx, by likewise.  Along a periodic axis only the regions that lie inside the domain (no wrap),
// along the others all of them.  nbx = 0: none (small grids), the blocked kernel does everything.
JacobiQuadPlan jacobi_quad_plan(const Grid &g, int ns, float k2)
{
    JacobiQuadPlan pl = {};
    if (ns != 5) return pl;                                  // instantiated for the sweep count of every configuration
    if (!(k2 >= 1e-3f && k2 <= 1e6f)) return pl;             // the kernel divides the update by 2 alpha/dx^2
    const int ot = R - 2 * ns;
    if (g.nx < R || g.ny < R) return pl;
    int lo[2], hi[2];
    const int n[2] = { g.nx, g.ny };
    for (int a = 0; a < 2; ++a) {
        if (g.bc[2 * a] == 0) {                              // periodic: origin >= 0 and end <= n
            lo[a] = (ns + ot - 1) / ot;
            hi[a] = (n[a] - R + ns) / ot;
        } else {
            lo[a] = 0;
            hi[a] = (n[a] + ot - 1) / ot - 1;
        }
        if (hi[a] < lo[a]) return pl;
    }
    pl.bx0 = lo[0]; pl.by0 = lo[1];
    pl.nbx = hi[0] - lo[0] + 1; pl.nby = hi[1] - lo[1] + 1;
    // y not periodic: every y region is taken here, so the regions may be 24 rows apart (34-row boxes, WY)
    pl.nby_blocked = pl.nby;
    if (g.bc[2] != 0) { pl.wy = 1; pl.nby = (g.ny + ot + 1) / (ot + 2); }
    // z chunks: one per region unless the grid is too small to fill the machine
    // z chunks: enough CTAs to fill the machine, and chunks of at most 512 planes: CTAs are not synchronised with each
    // other, and the shorter their march the less neighbouring regions drift apart along z, i.e. the more of the
    // re-reads of a neighbour's planes hit L2 (measured at 1024^3, DRAM reads per launch: 22.3 GB with one chunk of 1024
    // planes, 18.7 GB with two of 512 at the same 10.4 ms, 16.8 GB with four of 256 at 10.6 ms; 12.9 GB algorithmic)
    const long long cols = (long long)pl.nbx * pl.nby;
    long long nch = (2LL * 148 + cols - 1) / cols;
    if (nch < (g.nz + 511) / 512) nch = (g.nz + 511) / 512;
    if (nch < 1) nch = 1;
    int zc = (int)((g.nz + nch - 1) / nch);
    if (zc < 8 * ns) zc = 8 * ns;
    static int force_zc = -1;                    // IGR_JACOBI_ZC=n: planes per z chunk (tuning)
    if (force_zc < 0) { const char *e = getenv("IGR_JACOBI_ZC"); force_zc = e ? atoi(e) : 0; }
    if (force_zc >= 8 * ns) zc = force_zc;
    if (zc > g.nz) zc = g.nz;
    pl.zc = zc;
    return pl;
}

void launch_jacobi_quad(const Grid &g, int storage, int ns, const JacobiQuadPlan &pl, void *sig_out, float k2,
                        const CUtensorMap *rmap, const CUtensorMap *bmap, const CUtensorMap *smap, cudaStream_t st)
{
    if (pl.nbx <= 0 || ns != 5) return;
    static int qr = -1;                          // IGR_JACOBI_QR=2|4: rows per thread (tuning)
    if (qr < 0) { const char *e = getenv("IGR_JACOBI_QR"); qr = (e && atoi(e) == 2) ? 2 : 4; }
#define IGR_JQ(TT)                                                                                   \
    do {                                                                                             \
        if (pl.wy) launch_quad<TT, 5, 4, true>(g, pl, sig_out, k2, *rmap, *bmap, *smap, st);         \
        else if (qr == 2) launch_quad<TT, 5, 2, false>(g, pl, sig_out, k2, *rmap, *bmap, *smap, st); \
        else launch_quad<TT, 5, 4, false>(g, pl, sig_out, k2, *rmap, *bmap, *smap, st);              \
    } while (0)
    if (storage == 0) IGR_JQ(float);
    else if (storage == 1) IGR_JQ(__half);
    else IGR_JQ(__nv_bfloat16);
#undef IGR_JQ
}
