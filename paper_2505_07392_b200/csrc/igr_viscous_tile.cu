// igr_viscous_tile.cu -- NEXT-1 for sm_100a: r[1..4] += -div F_visc, streaming form.
// Formulas and citations: igr_viscous.cuh.
//
// Same 2.5-D plan as the tiled RHS (igr_rhs_tile.cu): a CTA owns a 32 x 8 column of cells and marches
// along z.  The current xy-plane of (rho, m) and of the five in-plane stress components arrives with its
// 3-cell halo by TMA (two 4-D boxes per plane, 3-slot ring, issued three planes ahead); the z stencil of
// (rho, m, tau_xz, tau_yz, tau_zz) lives in a sliding register window fed by coalesced own-column loads
// issued one plane ahead of use.  Every face is evaluated once per CTA: x+ / y+ / z+ by the owning thread,
// x- by shuffle, y- through shared memory, z- from the previous step; the low-x and low-y tile edges by
// two designated warps.  One __syncthreads per plane (exchange buffers double-buffered by step parity).
#include "igr_viscous.cuh"
#include "igr_tma.cuh"

#include <type_traits>

namespace {

constexpr int TX = 32, TY = 8, NT = TX * TY;
constexpr int NSLOT = 3;

using namespace igr_tma;

template <typename T>
struct VTile {
    static constexpr int HX = 16 / (int)sizeof(T);        // x halo of the q box: 16 B
    static constexpr int BX = TX + 2 * HX, BY = TY + 6, PE = BX * BY;
    static constexpr int HXT = 4, BXT = TX + 2 * HXT, PET = BXT * BY;   // tau box (fp32)
    static constexpr int QBYTES = (4 * PE * (int)sizeof(T) + 127) / 128 * 128;
    static constexpr int TBYTES = (5 * PET * 4 + 127) / 128 * 128;
    static constexpr int SLOT = QBYTES + TBYTES;
    static constexpr int TXBYTES = 4 * PE * (int)sizeof(T) + 5 * PET * 4;
    static constexpr int FY_OFF = NSLOT * SLOT;                       // float [2][4][TY][TX]
    static constexpr int EX_OFF = FY_OFF + 2 * 4 * TY * TX * 4;       // float [2][4][TY]
    static constexpr int EY_OFF = EX_OFF + 2 * 4 * TY * 4;            // float [2][4][TX]
    static constexpr int BAR_OFF = (EY_OFF + 2 * 4 * TX * 4 + 7) / 8 * 8;
    static constexpr int TOTAL = BAR_OFF + NSLOT * 8;
};

template <typename T> __device__ __forceinline__ float lds(const T *p);
template <> __device__ __forceinline__ float lds<float>(const float *p) { return *p; }
template <> __device__ __forceinline__ float lds<__half>(const __half *p) { return __half2float(*p); }
template <> __device__ __forceinline__ float lds<__nv_bfloat16>(const __nv_bfloat16 *p) { return __bfloat162float(*p); }

}  // namespace

template <typename T, int ORDER, bool FUSE>
__global__ void __launch_bounds__(NT, 2)
k_viscous_tile(const __grid_constant__ CUtensorMap qmap, const __grid_constant__ CUtensorMap tmap, Grid g,
               ViscTileArgs a)
{
    using TL = VTile<T>;
    extern __shared__ __align__(1024) unsigned char smem[];
    float *FYbase = reinterpret_cast<float *>(smem + TL::FY_OFF);
    float *EXbase = reinterpret_cast<float *>(smem + TL::EX_OFF);
    float *EYbase = reinterpret_cast<float *>(smem + TL::EY_OFF);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + TL::BAR_OFF);

    const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5, warp = ty;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int kz0 = blockIdx.z * a.zc, nkz = min(a.zc, g.nz - kz0);
    const int i = x0 + tx, j = y0 + ty;
    const bool valid = (i < g.nx) && (j < g.ny);

    // plane p of this chunk <-> cell plane kz0 + p <-> padded z index kz0 + p + 3
    const int cxq = g.gx + x0 - TL::HX, cxt = g.gx + x0 - TL::HXT, cy = y0;
    auto issue = [&](int p, int slot) {
        unsigned char *dst = smem + slot * TL::SLOT;
        mbar_expect_tx(&full[slot], TL::TXBYTES);
        tma_load_4d(dst, &qmap, cxq, cy, kz0 + p + IGR_NG, 0, &full[slot]);
        tma_load_4d(dst + TL::QBYTES, &tmap, cxt, cy, kz0 + p + IGR_NG, 0, &full[slot]);
    };
    if (tid == 0) {
        for (int s = 0; s < NSLOT; ++s) mbar_init(&full[s], 1);
        fence_init();
        for (int p = 0; p < NSLOT && p < nkz; ++p) issue(p, p);
    }
    __syncthreads();

    // own column in global memory (columns beyond the domain are clamped into the padding: unused values)
    const unsigned col = (unsigned)(min(i, g.nx) + g.gx) + (unsigned)g.sy * (unsigned)(min(j, g.ny) + IGR_NG);
    const unsigned usz = (unsigned)g.sz;
    const unsigned colc = (unsigned)(min(i, g.nx - 1) + g.gx) + (unsigned)g.sy * (unsigned)(min(j, g.ny - 1) + IGR_NG);
    const T *qf[4] = { (const T *)a.q[0], (const T *)a.q[1], (const T *)a.q[2], (const T *)a.q[3] };
    const float *tz[3] = { a.tau + (size_t)IGR_TAU_XZ * g.np, a.tau + (size_t)IGR_TAU_YZ * g.np,
                           a.tau + (size_t)IGR_TAU_ZZ * g.np };
    auto fetch = [&](int k, float out[7]) {                       // cell plane k in [-3, nz + 2]
        const unsigned id = col + usz * (unsigned)(min(k, g.nz + IGR_NG - 1) + IGR_NG);
#pragma unroll
        for (int f = 0; f < 4; ++f) out[f] = ldf(qf[f] + id);
#pragma unroll
        for (int f = 0; f < 3; ++f) out[4 + f] = tz[f][id];
    };

    // ---- prologue: window of cells kz0-3 .. kz0+2, H of the face kz0-1/2
    float W[7][6];
    {
        float v[7];
#pragma unroll
        for (int s = 0; s < 6; ++s) {
            fetch(kz0 - 3 + s, v);
#pragma unroll
            for (int f = 0; f < 7; ++f) W[f][s] = v[f];
        }
    }
    float Hz_prev[4];
    igr_visc::face<ORDER>(W, W + 4, Hz_prev);
#pragma unroll
    for (int f = 0; f < 7; ++f) {
#pragma unroll
        for (int s = 0; s < 5; ++s) W[f][s] = W[f][s + 1];
    }
    float pre[7];
    fetch(kz0 + 3, pre);

    const int ownq = (3 + ty) * TL::BX + TL::HX + tx;
    const int ownt = (3 + ty) * TL::BXT + TL::HXT + tx;
    int slot = 0, phase = 0;
    float vmax = 0.f;
    bool bad = false;
    for (int t = 0; t < nkz; ++t) {
#pragma unroll
        for (int f = 0; f < 7; ++f) W[f][5] = pre[f];
        fetch(kz0 + t + 4, pre);                                   // lands during this step
        const unsigned id = colc + usz * (unsigned)(kz0 + t + IGR_NG);   // clamped column: reads are always valid
        float r_pre[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) r_pre[c] = a.r[1 + c][id];
        // fused update: everything the epilogue reads pointwise is fetched now
        float r0 = 0.f, Es = 0.f, qn_pre[5];
        if (FUSE) {
            r0 = a.r[0][id]; Es = ldf(reinterpret_cast<const T *>(a.q[4]) + id);
            if (a.read_qn) {
#pragma unroll
                for (int c = 0; c < 5; ++c) qn_pre[c] = ldf(reinterpret_cast<const T *>(a.qn[c]) + id);
            }
        }

        mbar_wait(&full[slot], phase);
        const T *qc = reinterpret_cast<const T *>(smem + slot * TL::SLOT);
        const float *tc = reinterpret_cast<const float *>(smem + slot * TL::SLOT + TL::QBYTES);
        float *FY = FYbase + (t & 1) * 4 * TY * TX, *EX = EXbase + (t & 1) * 4 * TY, *EY = EYbase + (t & 1) * 4 * TX;

        float Hx[4], Hy[4];
        {   // x+ face: cells i-2 .. i+3
            float tq[4][6], tt[3][6];
#pragma unroll
            for (int f = 0; f < 4; ++f) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tq[f][s] = (s == 2) ? W[f][2] : lds<T>(qc + f * TL::PE + ownq + (s - 2));
            }
#pragma unroll
            for (int aa = 0; aa < 3; ++aa) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tt[aa][s] = tc[igr_visc::tau_field(0, aa) * TL::PET + ownt + (s - 2)];
            }
            igr_visc::face<ORDER>(tq, tt, Hx);
        }
        {   // y+ face: cells j-2 .. j+3
            float tq[4][6], tt[3][6];
#pragma unroll
            for (int f = 0; f < 4; ++f) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tq[f][s] = (s == 2) ? W[f][2] : lds<T>(qc + f * TL::PE + ownq + (s - 2) * TL::BX);
            }
#pragma unroll
            for (int aa = 0; aa < 3; ++aa) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tt[aa][s] = tc[igr_visc::tau_field(1, aa) * TL::PET + ownt + (s - 2) * TL::BXT];
            }
            igr_visc::face<ORDER>(tq, tt, Hy);
#pragma unroll
            for (int c = 0; c < 4; ++c) FY[(c * TY + ty) * TX + tx] = Hy[c];
        }
        if (warp == 2 && tx < TY) {
            // faces on the tile's low-x edge: between box columns HX-1 | HX of row tx
            float tq[4][6], tt[3][6], He[4];
            const int bq = (3 + tx) * TL::BX + TL::HX - 1, bt = (3 + tx) * TL::BXT + TL::HXT - 1;
#pragma unroll
            for (int f = 0; f < 4; ++f) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tq[f][s] = lds<T>(qc + f * TL::PE + bq + (s - 2));
            }
#pragma unroll
            for (int aa = 0; aa < 3; ++aa) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tt[aa][s] = tc[igr_visc::tau_field(0, aa) * TL::PET + bt + (s - 2)];
            }
            igr_visc::face<ORDER>(tq, tt, He);
#pragma unroll
            for (int c = 0; c < 4; ++c) EX[c * TY + tx] = He[c];
        }
        if (warp == 3) {
            // faces on the tile's low-y edge: between box rows 2 | 3 of column tx
            float tq[4][6], tt[3][6], He[4];
            const int bq = 2 * TL::BX + TL::HX + tx, bt = 2 * TL::BXT + TL::HXT + tx;
#pragma unroll
            for (int f = 0; f < 4; ++f) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tq[f][s] = lds<T>(qc + f * TL::PE + bq + (s - 2) * TL::BX);
            }
#pragma unroll
            for (int aa = 0; aa < 3; ++aa) {
#pragma unroll
                for (int s = 0; s < 6; ++s) tt[aa][s] = tc[igr_visc::tau_field(1, aa) * TL::PET + bt + (s - 2) * TL::BXT];
            }
            igr_visc::face<ORDER>(tq, tt, He);
#pragma unroll
            for (int c = 0; c < 4; ++c) EY[c * TX + tx] = He[c];
        }
        __syncthreads();                                    // the only barrier of the step
        if (tid == 0 && t + NSLOT < nkz) {                  // the slot of this plane is free again
            fence_async();
            issue(t + NSLOT, slot);
        }

        float Hz[4], rr[5];
        igr_visc::face<ORDER>(W, W + 4, Hz);
        rr[0] = r0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            float hxm = __shfl_up_sync(0xffffffffu, Hx[c], 1);
            if (tx == 0) hxm = EX[c * TY + ty];
            const float hym = (ty == 0) ? EY[c * TX + tx] : FY[(c * TY + ty - 1) * TX + tx];
            float acc = __fsub_rn(Hx[c], hxm);
            acc = __fadd_rn(acc, __fsub_rn(Hy[c], hym));
            acc = __fadd_rn(acc, __fsub_rn(Hz[c], Hz_prev[c]));
            Hz_prev[c] = Hz[c];
            rr[1 + c] = __fmaf_rn(a.inv_dx, acc, r_pre[c]);
            if (!FUSE && valid) a.r[1 + c][id] = rr[1 + c];
        }
        if (FUSE && valid) {
            float o[5];
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                const float qs = (c < 4) ? W[c][2] : Es;
                const float qn = a.read_qn ? qn_pre[c] : qs;
                o[c] = __fmaf_rn(a.beta, __fmaf_rn(a.dt, rr[c], __fsub_rn(qs, qn)), qn);
                stf(reinterpret_cast<T *>(a.qout[c]) + id, o[c]);
            }
            if (a.wave && kz0 + t >= g.wk0 && kz0 + t < g.wk1) {
                if (sizeof(T) < 4) {
#pragma unroll
                    for (int c = 0; c < 5; ++c) o[c] = ldf(reinterpret_cast<const T *>(a.qout[c]) + id);
                }
                vmax = fmaxf(vmax, wavespeed_of(o[0], o[1], o[2], o[3], o[4], a.gamma, bad));
            }
        }
#pragma unroll
        for (int f = 0; f < 7; ++f) {
#pragma unroll
            for (int s = 0; s < 5; ++s) W[f][s] = W[f][s + 1];
        }
        if (++slot == NSLOT) { slot = 0; phase ^= 1; }
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

template <typename T, int ORDER, bool FUSE>
void launch_one(const Grid &g, const CUtensorMap &qmap, const CUtensorMap &tmap, ViscTileArgs a, cudaStream_t st)
{
    using TL = VTile<T>;
    static bool configured = false;
    if (!configured) {
        cudaFuncSetAttribute(k_viscous_tile<T, ORDER, FUSE>, cudaFuncAttributeMaxDynamicSharedMemorySize, TL::TOTAL);
        configured = true;
    }
    dim3 grid((g.nx + TX - 1) / TX, (g.ny + TY - 1) / TY, (g.nz + a.zc - 1) / a.zc);
    k_viscous_tile<T, ORDER, FUSE><<<grid, NT, TL::TOTAL, st>>>(qmap, tmap, g, a);
}

}  // namespace

int visc_tile_make_maps(const Grid &g, int storage, const StagePtrs st[3], int n_state, const float *tau,
                        ViscTileMaps *out, const char **err)
{
    out->valid = false;
    if (!igr_tma::get_encode()) { *err = "cuTensorMapEncodeTiled entry point not available"; return 1; }
    const size_t es = storage == 0 ? 4 : 2;
    const cuuint32_t bx = TX + 2 * (16 / (cuuint32_t)es), by = TY + 6;
    for (int b = 0; b < 3; ++b) {
        const StagePtrs &s = st[b < n_state ? b : n_state - 1];
        const cuuint64_t fstride = (cuuint64_t)((char *)s.f[1] - (char *)s.f[0]);
        for (int f = 1; f < 4; ++f)
            if ((cuuint64_t)((char *)s.f[f] - (char *)s.f[f - 1]) != fstride) {
                *err = "state fields are not equally spaced"; return 2;
            }
        cuuint64_t dims[4] = { (cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz, 4 };
        cuuint64_t strides[3] = { (cuuint64_t)g.px * es, (cuuint64_t)g.px * g.py * es, fstride };
        cuuint32_t box[4] = { bx, by, 1, 4 };
        if (!igr_tma::encode(&out->q[b], igr_tma::data_type(storage), 4, s.f[0], dims, strides, box)) {
            *err = "cuTensorMapEncodeTiled(q, viscous) failed"; return 3;
        }
    }
    {
        cuuint64_t dims[4] = { (cuuint64_t)g.px, (cuuint64_t)g.py, (cuuint64_t)g.pz, 5 };
        cuuint64_t strides[3] = { (cuuint64_t)g.px * 4, (cuuint64_t)g.px * g.py * 4, (cuuint64_t)g.np * 4 };
        cuuint32_t box[4] = { TX + 8, by, 1, 5 };
        if (!igr_tma::encode(&out->tau, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, tau, dims, strides, box)) {
            *err = "cuTensorMapEncodeTiled(tau) failed"; return 3;
        }
    }
    out->valid = true;
    return 0;
}

void launch_viscous_tile(const Grid &g, int storage, int order, bool fused, const CUtensorMap &qmap,
                         const CUtensorMap &tmap, ViscTileArgs a, cudaStream_t st)
{
    if (a.zc <= 0) {
        // about 4 waves of 148 SMs x 2 CTAs, chunks of at least 32 planes
        const long long cols = (long long)((g.nx + TX - 1) / TX) * ((g.ny + TY - 1) / TY);
        long long nch = (4LL * 148 * 2 + cols - 1) / cols;
        int zc = (int)((g.nz + nch - 1) / nch);
        if (zc < 32) zc = 32;
        if (zc > g.nz) zc = g.nz;
        a.zc = zc;
    }
#define IGR_VCASE(TT)                                                                              \
    do {                                                                                           \
        if (order == 5) { if (fused) launch_one<TT, 5, true>(g, qmap, tmap, a, st); else launch_one<TT, 5, false>(g, qmap, tmap, a, st); } \
        else { if (fused) launch_one<TT, 3, true>(g, qmap, tmap, a, st); else launch_one<TT, 3, false>(g, qmap, tmap, a, st); }            \
    } while (0)
    if (storage == 0) IGR_VCASE(float);
    else if (storage == 1) IGR_VCASE(__half);
    else IGR_VCASE(__nv_bfloat16);
#undef IGR_VCASE
}
