// igr_api.cu -- the C ABI of libigr.so (include/igr.h): solver object, buffer carving, host<->device
// marshalling and the sequencing of the kernels of one SSP-RK3 step.  No arithmetic of the method
// is done on the host except the fp64 evaluation of the inflow blend weights at creation.
#include "../../include/igr.h"
#include "igr_kernels.h"
#include "igr_rhs_tile.cuh"
#include "igr_viscous.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

namespace {

constexpr size_t kAlign = 256;
constexpr size_t kStageBytes = 64u << 20;          // staging buffer for host <-> device copies

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline size_t elem_size(int storage) { return storage == IGR_STORE_F64 ? 8 : (storage == IGR_STORE_F32 ? 4 : 2); }

Grid make_grid(int nx, int ny, int nz, int storage, const int32_t *faces)
{
    Grid g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    const int per32 = (int)(32 / elem_size(storage));     // elements per 32 bytes
    g.gx = per32;                                         // 8 (fp32) or 16 (half): >= 3 ghosts
    g.px = (int)align_up((size_t)nx + 2 * g.gx, per32);
    g.py = ny + 2 * IGR_NG;
    g.pz = nz + 2 * IGR_NG;
    g.sy = g.px;
    g.sz = (long long)g.px * g.py;
    g.np = g.sz * g.pz;
    for (int f = 0; f < 6; ++f) g.bc[f] = faces ? faces[f] : 0;
    g.wk0 = 0; g.wk1 = nz;
    return g;
}

struct Layout {
    size_t q_bytes, f_bytes;        // one padded field in storage type / in fp32
    int n_state;                    // state buffers (2 unfused, 3 fused)
    int n_r;                        // r fields inside the workspace (5, or 0: allocated on first use)
    size_t total;
};

Layout make_layout(const Grid &g, int storage, int fused, int variant, int nf = 5)
{
    Layout L;
    L.q_bytes = align_up((size_t)g.np * elem_size(storage), kAlign);
    L.f_bytes = align_up((size_t)g.np * (storage == IGR_STORE_F64 ? 8 : 4), kAlign);   // b, r: fp32 (fp64 mode: fp64)
    L.n_state = fused ? 3 : 2;
    // the fused tiled step never materialises r: it is allocated only if an unfused row, igr_get_rhs or
    // the viscous path asks for it (5 fp32 fields less: 18 instead of 23 fields at rest)
    L.n_r = (fused && variant == IGR_VARIANT_TILED) ? 0 : 5;
    // states + Sigma x2 (storage type) + b + r[n_r] (fp32) + staging + wave result (+ the mixture density with
    // two fluids)
    L.total = (size_t)L.n_state * nf * L.q_bytes + 2 * L.q_bytes + (1 + L.n_r + (nf == 7 ? 1 : 0)) * L.f_bytes +
              kStageBytes + kAlign;
    return L;
}

}  // namespace

struct igr_solver {
    Grid g;
    int storage = 0, fused = 0, variant = 0, order = 5, n_jacobi = 5;
    RhsTileMaps maps;
    SourceMaps smaps[3];             // TMA maps of the source kernel, one set per state buffer
    JacobiMaps jmaps;                // TMA maps of the blocked Jacobi kernel (32-row boxes)
    JacobiMaps jmaps2;               // the same with 34-row boxes (quad regions 24 rows apart)
    double dx = 0, gamma = 0, alpha = 0;
    int nf = 5;                      // conserved fields: 5, or 7 with two fluids (NEXT-3, reading A21)
    double gamma2 = 0;               // two fluids: exponent of fluid 2
    float *rhot = nullptr;           // two fluids: mixture density of every padded cell (fp32)
    cudaStream_t stream = nullptr;
    char *base = nullptr;            // device memory (owned or caller's workspace)
    bool owns_base = false;
    StagePtrs st[3];                 // state buffers: st[cur] is the current stage buffer
    int cur = 0;                     // index of the buffer holding q^n / the current state
    void *sig[2] = { nullptr, nullptr };
    int sig_cur = 0;
    float *b = nullptr;
    float *r[5] = { nullptr, nullptr, nullptr, nullptr, nullptr };
    float *stage = nullptr;          // staging, kStageBytes
    WaveResult *wave = nullptr;      // device
    bool wave_valid = false;         // wave holds the wave speed of the current state
    BcDesc bc;
    Inflow64 bc64;                   // fp64 mode: the same tables in double
    std::vector<void *> bc_allocs;   // device arrays of the inflow faces
    std::string err;
    double mu = 0, zeta = 0;         // viscosity (NEXT-1); 0, 0: inviscid
    float *r_owned = nullptr;        // r[5] when it is not part of the workspace (ensure_r)
    float *tau = nullptr;            // six stress fields (allocated by igr_set_viscosity; igr_viscous.cuh)
    ViscTileMaps vmaps;              // TMA maps of the tiled viscous kernel
    struct Neighbor {                // NEXT-2: neighbouring slab on z- / z+ (igr_set_neighbor)
        bool active = false;
        igr_export desc;
        const char *base = nullptr;  // the neighbour's allocation as addressable from this process
        int dst = 0, src = 0, count = 0;
    } nb[2];
    cudaEvent_t ipc_ev[2] = { nullptr, nullptr };   // interprocess events: stage complete / pulls complete
    long long launches = 0;          // kernels launched so far (igr_kernel_launches)
    bool profile = false;            // per-row CUDA-event timing (igr_profile)
    std::vector<cudaEvent_t> ev;     // start/stop pairs
    std::vector<int> ev_row;

    int fail(int code, const char *what, cudaError_t e = cudaSuccess)
    {
        char buf[512];
        if (e != cudaSuccess) snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
        else snprintf(buf, sizeof buf, "%s", what);
        err = buf;
        return code;
    }
};

static_assert(IGR_BC_EXTERNAL == kBcExternal, "igr.h and igr_common.cuh disagree");

namespace {

// fp64 evaluation of the inflow blend weight (igr.h, igr_patch; reading A8b)
double patch_weight(const igr_patch &p, int t0, int t1)
{
    const double d0 = (t0 + 0.5) - p.c0, d1 = (t1 + 0.5) - p.c1;
    const double r2 = d0 * d0 + d1 * d1;
    if (p.edge <= 0.0) return r2 <= p.radius * p.radius ? 1.0 : 0.0;
    const double r = std::sqrt(r2);
    if (r >= p.radius + 4.0 * p.edge) return 0.0;
    return 0.5 * (1.0 - std::tanh((r - p.radius) / p.edge));
}

int build_inflow(igr_solver *s, const igr_bc *bc)
{
    const int n[3] = { s->g.nx, s->g.ny, s->g.nz };
    for (int f = 0; f < 6; ++f) {
        InflowFace &F = s->bc.inflow[f];
        F.weight = nullptr; F.fixed = nullptr; F.n0 = F.n1 = 0;
        s->bc64.weight[f] = nullptr; s->bc64.fixed[f] = nullptr; s->bc64.n0[f] = s->bc64.n1[f] = 0;
        if (bc->face[f] != IGR_BC_INFLOW || bc->n_patches[f] <= 0) continue;
        if (!bc->patches[f]) return s->fail(IGR_ERR_ARG, "igr_create: inflow face without patches array");
        const int a = f / 2;
        F.n0 = (a == 0) ? n[1] : n[0];
        F.n1 = (a == 2) ? n[1] : n[2];
        const int nf = s->nf;
        std::vector<float> w((size_t)F.n0 * F.n1), fx((size_t)F.n0 * F.n1 * nf, 0.f);
        std::vector<double> w64, fx64;
        if (s->storage == IGR_STORE_F64) { w64.assign(w.size(), 0.0); fx64.assign(fx.size(), 0.0); }
        for (int t1 = 0; t1 < F.n1; ++t1)
            for (int t0 = 0; t0 < F.n0; ++t0) {
                double best = 0.0; const igr_patch *bp = nullptr;
                for (int m = 0; m < bc->n_patches[f]; ++m) {
                    double ww = patch_weight(bc->patches[f][m], t0, t1);
                    if (ww > best) { best = ww; bp = &bc->patches[f][m]; }
                }
                const size_t id = (size_t)t1 * F.n0 + t0;
                w[id] = (float)best;
                if (best >= 1.0) w[id] = 1.0f;
                else if (best > 0.0 && w[id] >= 1.0f) w[id] = 0.99999994f;   // keep "w < 1" in fp32
                if (bp && nf == 5) {
                    const double ke = 0.5 * bp->rho * (bp->u * bp->u + bp->v * bp->v + bp->w * bp->w);
                    const double v[5] = { bp->rho, bp->rho * bp->u, bp->rho * bp->v, bp->rho * bp->w,
                                          bp->p / (s->gamma - 1.0) + ke };
                    for (int c = 0; c < 5; ++c) fx[id * 5 + c] = (float)v[c];
                    if (!w64.empty()) { w64[id] = best; for (int c = 0; c < 5; ++c) fx64[id * 5 + c] = v[c]; }
                } else if (bp) {             // two fluids (igr.h, igr_patch): rho = fluid 1, rho2 = fluid 2
                    const double m1 = bp->a1 * bp->rho, m2 = (1.0 - bp->a1) * bp->rho2, rm = m1 + m2;
                    const double ke = 0.5 * rm * (bp->u * bp->u + bp->v * bp->v + bp->w * bp->w);
                    const double G = bp->a1 / (s->gamma - 1.0) + (1.0 - bp->a1) / (s->gamma2 - 1.0);
                    const double v[7] = { m1, m2, rm * bp->u, rm * bp->v, rm * bp->w, bp->p * G + ke, bp->a1 };
                    for (int c = 0; c < 7; ++c) fx[id * 7 + c] = (float)v[c];
                }
            }
        float *dw = nullptr, *dfx = nullptr;
        if (cudaMalloc(&dw, w.size() * 4) != cudaSuccess || cudaMalloc(&dfx, fx.size() * 4) != cudaSuccess)
            return s->fail(IGR_ERR_ALLOC, "igr_create: cudaMalloc of inflow tables failed");
        s->bc_allocs.push_back(dw); s->bc_allocs.push_back(dfx);
        IGR_CUDA_OK(cudaMemcpy(dw, w.data(), w.size() * 4, cudaMemcpyHostToDevice));
        IGR_CUDA_OK(cudaMemcpy(dfx, fx.data(), fx.size() * 4, cudaMemcpyHostToDevice));
        F.weight = dw; F.fixed = dfx;
        if (!w64.empty()) {
            double *dw64 = nullptr, *dfx64 = nullptr;
            if (cudaMalloc(&dw64, w64.size() * 8) != cudaSuccess || cudaMalloc(&dfx64, fx64.size() * 8) != cudaSuccess)
                return s->fail(IGR_ERR_ALLOC, "igr_create: cudaMalloc of inflow tables failed");
            s->bc_allocs.push_back(dw64); s->bc_allocs.push_back(dfx64);
            IGR_CUDA_OK(cudaMemcpy(dw64, w64.data(), w64.size() * 8, cudaMemcpyHostToDevice));
            IGR_CUDA_OK(cudaMemcpy(dfx64, fx64.data(), fx64.size() * 8, cudaMemcpyHostToDevice));
            s->bc64.weight[f] = dw64; s->bc64.fixed[f] = dfx64; s->bc64.n0[f] = F.n0; s->bc64.n1[f] = F.n1;
        }
    }
    return IGR_OK;
}

bool is_device_pointer(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// copy one user field (interior, fp32, host or device) into / out of a padded field
// (planes [kfirst, kfirst + nplanes) of the field; `user` holds exactly those planes; nplanes < 0: all)
// `ubytes`: element size of the user array (4: fp32, the ABI's default; 8: the *_f64 calls of the fp64 mode)
int field_in(igr_solver *s, const void *user, void *field, int storage, int kfirst = 0, int nplanes = -1, int ubytes = 4)
{
    const Grid &g = s->g;
    if (nplanes < 0) nplanes = g.nz;
    auto unpack = [&](const void *src, int k0, int nk) {
        if (storage == IGR_STORE_F64) launch64_unpack(g, src, ubytes == 4, (double *)field, k0, nk, s->stream);
        else launch_unpack_field(g, storage, (const float *)src, field, k0, nk, s->stream);
    };
    if (storage != IGR_STORE_F64 && ubytes != 4) return s->fail(IGR_ERR_ARG, "fp64 arrays: only with IGR_STORE_F64");
    if (is_device_pointer(user)) {
        unpack(user, kfirst, nplanes);
        return IGR_OK;
    }
    const size_t plane = (size_t)g.nx * g.ny * ubytes;
    int chunk = (int)(kStageBytes / plane);
    if (chunk < 1) return s->fail(IGR_ERR_ARG, "igr: one z-plane exceeds the staging buffer");
    for (int k0 = 0; k0 < nplanes; k0 += chunk) {
        const int nk = (nplanes - k0 < chunk) ? nplanes - k0 : chunk;
        IGR_CUDA_OK(cudaMemcpyAsync(s->stage, (const char *)user + (size_t)k0 * plane, nk * plane,
                                    cudaMemcpyHostToDevice, s->stream));
        unpack(s->stage, kfirst + k0, nk);
        // the staging buffer is reused by the next chunk and `user` is borrowed for the duration of the call
        // only (igr.h): the copy must have left the host buffer before this returns
        IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    }
    return IGR_OK;
}

int field_out(igr_solver *s, const void *field, void *user, int storage, int kfirst = 0, int nplanes = -1, int ubytes = 4)
{
    const Grid &g = s->g;
    if (nplanes < 0) nplanes = g.nz;
    auto pack = [&](void *dst, int k0, int nk) {
        if (storage == IGR_STORE_F64) launch64_pack(g, (const double *)field, dst, ubytes == 4, k0, nk, s->stream);
        else launch_pack_field(g, storage, field, (float *)dst, k0, nk, s->stream);
    };
    if (storage != IGR_STORE_F64 && ubytes != 4) return s->fail(IGR_ERR_ARG, "fp64 arrays: only with IGR_STORE_F64");
    if (is_device_pointer(user)) {
        pack(user, kfirst, nplanes);
        return IGR_OK;
    }
    const size_t plane = (size_t)g.nx * g.ny * ubytes;
    int chunk = (int)(kStageBytes / plane);
    if (chunk < 1) return s->fail(IGR_ERR_ARG, "igr: one z-plane exceeds the staging buffer");
    for (int k0 = 0; k0 < nplanes; k0 += chunk) {
        const int nk = (nplanes - k0 < chunk) ? nplanes - k0 : chunk;
        pack(s->stage, kfirst + k0, nk);
        IGR_CUDA_OK(cudaMemcpyAsync((char *)user + (size_t)k0 * plane, s->stage, nk * plane,
                                    cudaMemcpyDeviceToHost, s->stream));
        IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    }
    return IGR_OK;
}

// times one row of the hot path with a CUDA-event pair on the solver's stream when profiling is on
struct RowTimer {
    igr_solver *s; int row;
    RowTimer(igr_solver *s_, int row_, int n_launch) : s(s_), row(row_)
    {
        s->launches += n_launch;
        if (!s->profile) return;
        cudaEvent_t a, b;
        cudaEventCreate(&a); cudaEventCreate(&b);
        s->ev.push_back(a); s->ev.push_back(b); s->ev_row.push_back(row);
        cudaEventRecord(a, s->stream);
    }
    ~RowTimer() { if (s->profile) cudaEventRecord(s->ev.back(), s->stream); }
};

// r[5] of a fused tiled solver is not part of the workspace: allocate it on first use
int ensure_r(igr_solver *s)
{
    if (s->r[0]) return IGR_OK;
    const size_t fb = align_up((size_t)s->g.np * 4, kAlign);
    if (cudaMalloc((void **)&s->r_owned, 5 * fb) != cudaSuccess) {
        cudaGetLastError();
        s->r_owned = nullptr;
        return s->fail(IGR_ERR_ALLOC, "cudaMalloc of the RHS fields failed");
    }
    IGR_CUDA_OK(cudaMemsetAsync(s->r_owned, 0, 5 * fb, s->stream));
    for (int c = 0; c < 5; ++c) s->r[c] = (float *)((char *)s->r_owned + c * fb);
    return IGR_OK;
}

int finish(igr_solver *s, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return s->fail(IGR_ERR_CUDA, what, e);
    return IGR_OK;
}

}  // namespace

// ===================================================================================== C ABI
extern "C" {

size_t igr_workspace_bytes(int nx, int ny, int nz, const igr_options *opt)
{
    if (nx < 1 || ny < 1 || nz < 1) return 0;
    const int storage = opt ? opt->storage : IGR_STORE_F32;
    const int fused = (opt && storage != IGR_STORE_F64) ? opt->fused : (storage == IGR_STORE_F64 ? 0 : 1);
    if (storage < 0 || storage > 3) return 0;
    Grid g = make_grid(nx, ny, nz, storage, nullptr);
    return make_layout(g, storage, fused, storage == IGR_STORE_F64 ? IGR_VARIANT_SIMPLE : (opt ? opt->variant : 0),
                       (opt && opt->n_fluids == 2) ? 7 : 5).total;
}

int igr_create(int nx, int ny, int nz, double dx, double gamma, double alpha, int order,
               int n_jacobi, const igr_bc *bc, igr_solver **out)
{
    return igr_create_ex(nx, ny, nz, dx, gamma, alpha, order, n_jacobi, bc, nullptr, out);
}

int igr_create_ex(int nx, int ny, int nz, double dx, double gamma, double alpha, int order,
                  int n_jacobi, const igr_bc *bc, const igr_options *opt, igr_solver **out)
{
    if (!out) return IGR_ERR_ARG;
    *out = nullptr;
    if (!bc || nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(gamma > 1) || !(alpha >= 0) ||
        n_jacobi < 0 || (order != 5 && order != 3))
        return IGR_ERR_ARG;
    const int storage = opt ? opt->storage : IGR_STORE_F32;
    if (storage < 0 || storage > 3) return IGR_ERR_ARG;
    for (int a = 0; a < 3; ++a) {
        const int lo = bc->face[2 * a], hi = bc->face[2 * a + 1];
        if (lo < 0 || lo > 3 || hi < 0 || hi > 3) return IGR_ERR_BC;
        if ((lo == IGR_BC_PERIODIC) != (hi == IGR_BC_PERIODIC)) return IGR_ERR_BC;
        if (a < 2 && (lo == IGR_BC_EXTERNAL || hi == IGR_BC_EXTERNAL)) return IGR_ERR_BC;   // z slabs only
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return IGR_ERR_CUDA; }

    const bool two = opt && opt->n_fluids == 2;
    if (opt && (opt->n_fluids < 0 || opt->n_fluids > 2)) return IGR_ERR_ARG;
    // two fluids (NEXT-3): fp32 storage, order 5, fused tiled kernels only
    if (two && (storage != IGR_STORE_F32 || order != 5 || !opt->fused || opt->variant != IGR_VARIANT_TILED ||
                !(opt->gamma2 > 1)))
        return IGR_ERR_ARG;

    igr_solver *s = new igr_solver();
    s->nf = two ? 7 : 5;
    s->gamma2 = two ? opt->gamma2 : 0.0;
    s->storage = storage;
    s->fused = opt ? (opt->fused != 0) : 1;                 // igr_create: the fused (headline) path
    s->variant = opt ? opt->variant : 0;
    if (storage == IGR_STORE_F64) {                         // fp64 mode: one kernel per row, r materialised
        if (two) { delete s; return IGR_ERR_ARG; }
        s->fused = 0; s->variant = IGR_VARIANT_SIMPLE;
    }
    s->maps.valid = false;
    s->jmaps.valid = false;
    s->jmaps2.valid = false;
    for (int b = 0; b < 3; ++b) s->smaps[b].valid = false;
    s->order = order; s->n_jacobi = n_jacobi;
    s->dx = dx; s->gamma = gamma; s->alpha = alpha;
    s->stream = opt ? (cudaStream_t)opt->stream : nullptr;
    s->g = make_grid(nx, ny, nz, storage, bc->face);
    if (s->g.np > (long long)UINT32_MAX) {       // the kernels address cells with 32-bit unsigned element offsets
        delete s;
        return IGR_ERR_ARG;
    }
    const Layout L = make_layout(s->g, storage, s->fused, s->variant, s->nf);
    if (opt && opt->workspace) {
        if (opt->workspace_bytes < L.total || ((uintptr_t)opt->workspace % kAlign) != 0) {
            delete s;
            return IGR_ERR_ALLOC;
        }
        s->base = (char *)opt->workspace;
    } else {
        if (cudaMalloc((void **)&s->base, L.total) != cudaSuccess) {
            cudaGetLastError();
            delete s;
            return IGR_ERR_ALLOC;
        }
        s->owns_base = true;
    }
    // ghosts and the x padding must hold finite numbers: zero everything once
    if (cudaMemsetAsync(s->base, 0, L.total, s->stream) != cudaSuccess) { igr_destroy(s); return IGR_ERR_CUDA; }
    char *p = s->base;
    for (int b = 0; b < L.n_state; ++b)
        for (int c = 0; c < s->nf; ++c) { s->st[b].f[c] = p; p += L.q_bytes; }
    if (L.n_state < 3) s->st[2] = s->st[1];
    s->sig[0] = p; p += L.q_bytes;
    s->sig[1] = p; p += L.q_bytes;
    s->b = (float *)p; p += L.f_bytes;
    if (two) { s->rhot = (float *)p; p += L.f_bytes; }
    for (int c = 0; c < L.n_r; ++c) { s->r[c] = (float *)p; p += L.f_bytes; }
    s->stage = (float *)p; p += kStageBytes;
    s->wave = (WaveResult *)p;
    int rc = build_inflow(s, bc);
    if (rc != IGR_OK) { igr_destroy(s); return rc; }
    if (s->variant == IGR_VARIANT_TILED) {
        const char *msg = "";
        if (rhs_tile_make_maps(s->g, storage, s->st, L.n_state, s->sig, s->nf, &s->maps, &msg) != 0) {
            igr_destroy(s);
            return IGR_ERR_CUDA;
        }
        for (int b = 0; b < 3; ++b) {        // (rho, m) of every state buffer for the source kernel
            const StagePtrs &sp = s->st[b < L.n_state ? b : L.n_state - 1];
            void *f4[4] = { two ? (void *)s->rhot : sp.f[0], sp.f[two ? 2 : 1], sp.f[two ? 3 : 2], sp.f[two ? 4 : 3] };
            if (source_make_maps(s->g, storage, f4, &s->smaps[b]) != 0) { igr_destroy(s); return IGR_ERR_CUDA; }
        }
        // the density the Sigma equation reads: field 0 of the state, or the mixture density (two fluids)
        StagePtrs rho_of[3];
        for (int b = 0; b < 3; ++b) { rho_of[b] = s->st[b]; if (two) rho_of[b].f[0] = s->rhot; }
        if (jacobi_make_maps(s->g, storage, rho_of, L.n_state, s->sig, s->b, &s->jmaps) != 0 ||
            jacobi_make_maps(s->g, storage, rho_of, L.n_state, s->sig, s->b, &s->jmaps2, 34) != 0) {
            igr_destroy(s);
            return IGR_ERR_CUDA;
        }
    }
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) { igr_destroy(s); return IGR_ERR_CUDA; }
    *out = s;
    return IGR_OK;
}

void igr_destroy(igr_solver *s)
{
    if (!s) return;
    cudaStreamSynchronize(s->stream);
    for (int i = 0; i < 2; ++i)
        if (s->ipc_ev[i]) cudaEventDestroy(s->ipc_ev[i]);
    if (s->tau) cudaFree(s->tau);
    if (s->r_owned) cudaFree(s->r_owned);
    for (void *p : s->bc_allocs) cudaFree(p);
    if (s->owns_base && s->base) cudaFree(s->base);
    delete s;
}

const char *igr_last_error(const igr_solver *s) { return s ? s->err.c_str() : "null solver"; }

int igr_sync(igr_solver *s)
{
    if (!s) return IGR_ERR_ARG;
    IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    return finish(s, "igr_sync");
}

static int set_state_any(igr_solver *s, const void *q, int ubytes)
{
    if (!s || !q) return IGR_ERR_ARG;
    const size_t n = (size_t)s->g.nx * s->g.ny * s->g.nz;
    s->cur = 0;
    for (int c = 0; c < s->nf; ++c) {
        int rc = field_in(s, (const char *)q + c * n * ubytes, s->st[0].f[c], s->storage, 0, -1, ubytes);
        if (rc != IGR_OK) return rc;
    }
    const size_t qb = (size_t)s->g.np * elem_size(s->storage);
    IGR_CUDA_OK(cudaMemsetAsync(s->sig[0], 0, qb, s->stream));     // "Sigma = 0 at t = 0"
    IGR_CUDA_OK(cudaMemsetAsync(s->sig[1], 0, qb, s->stream));
    s->sig_cur = 0;
    s->wave_valid = false;
    return finish(s, "igr_set_state");
}

int igr_set_state(igr_solver *s, const float *q) { return set_state_any(s, q, 4); }
int igr_set_state_f64(igr_solver *s, const double *q) { return set_state_any(s, q, 8); }

int igr_get_state_f64(igr_solver *s, double *q)
{
    if (!s || !q) return IGR_ERR_ARG;
    const size_t n = (size_t)s->g.nx * s->g.ny * s->g.nz;
    for (int c = 0; c < s->nf; ++c) {
        int rc = field_out(s, s->st[s->cur].f[c], q + c * n, s->storage, 0, -1, 8);
        if (rc != IGR_OK) return rc;
    }
    return igr_sync(s);
}

int igr_get_sigma_f64(igr_solver *s, double *f)
{
    if (!s || !f) return IGR_ERR_ARG;
    int rc = field_out(s, s->sig[s->sig_cur], f, s->storage, 0, -1, 8);
    if (rc != IGR_OK) return rc;
    return igr_sync(s);
}

int igr_set_state_planes(igr_solver *s, int k0, int nk, const float *q)
{
    if (!s || !q || k0 < 0 || nk < 1 || k0 + nk > s->g.nz) return IGR_ERR_ARG;
    if (s->cur != 0) return s->fail(IGR_ERR_ARG, "igr_set_state_planes: called in the middle of a step");
    const size_t n = (size_t)s->g.nx * s->g.ny * nk;
    for (int c = 0; c < s->nf; ++c) {
        int rc = field_in(s, q + c * n, s->st[0].f[c], s->storage, k0, nk);
        if (rc != IGR_OK) return rc;
    }
    s->wave_valid = false;
    return finish(s, "igr_set_state_planes");
}

int igr_get_state_planes(igr_solver *s, int k0, int nk, float *q)
{
    if (!s || !q || k0 < 0 || nk < 1 || k0 + nk > s->g.nz) return IGR_ERR_ARG;
    const size_t n = (size_t)s->g.nx * s->g.ny * nk;
    for (int c = 0; c < s->nf; ++c) {
        int rc = field_out(s, s->st[s->cur].f[c], q + c * n, s->storage, k0, nk);
        if (rc != IGR_OK) return rc;
    }
    return igr_sync(s);
}

int igr_get_state(igr_solver *s, float *q)
{
    if (!s || !q) return IGR_ERR_ARG;
    const size_t n = (size_t)s->g.nx * s->g.ny * s->g.nz;
    for (int c = 0; c < s->nf; ++c) {
        int rc = field_out(s, s->st[s->cur].f[c], q + c * n, s->storage);
        if (rc != IGR_OK) return rc;
    }
    return igr_sync(s);
}

int igr_set_sigma(igr_solver *s, const float *f)
{
    if (!s || !f) return IGR_ERR_ARG;
    int rc = field_in(s, f, s->sig[s->sig_cur], s->storage);
    if (rc != IGR_OK) return rc;
    if (s->storage == IGR_STORE_F64) launch64_halo_sigma(s->g, (double *)s->sig[s->sig_cur], s->stream);
    else launch_halo_sigma(s->g, s->storage, s->sig[s->sig_cur], s->stream);
    return finish(s, "igr_set_sigma");
}

int igr_get_sigma(igr_solver *s, float *f)
{
    if (!s || !f) return IGR_ERR_ARG;
    int rc = field_out(s, s->sig[s->sig_cur], f, s->storage);
    if (rc != IGR_OK) return rc;
    return igr_sync(s);
}

int igr_get_source(igr_solver *s, float *f)
{
    if (!s || !f) return IGR_ERR_ARG;
    if (s->storage == IGR_STORE_F64) return s->fail(IGR_ERR_ARG, "igr_get_source: not available in the fp64 mode");
    int rc = field_out(s, s->b, f, IGR_STORE_F32);
    if (rc != IGR_OK) return rc;
    return igr_sync(s);
}

int igr_set_source(igr_solver *s, const float *f)
{
    if (!s || !f) return IGR_ERR_ARG;
    if (s->storage == IGR_STORE_F64) return s->fail(IGR_ERR_ARG, "igr_set_source: not available in the fp64 mode");
    int rc = field_in(s, f, s->b, IGR_STORE_F32);
    if (rc != IGR_OK) return rc;
    return finish(s, "igr_set_source");
}

int igr_get_rhs(igr_solver *s, float *r)
{
    if (!s || !r) return IGR_ERR_ARG;
    if (s->nf != 5) return s->fail(IGR_ERR_ARG, "two fluids: r is never materialised (fused step only)");
    if (s->storage == IGR_STORE_F64) return s->fail(IGR_ERR_ARG, "igr_get_rhs: not available in the fp64 mode");
    { const int rc = ensure_r(s); if (rc != IGR_OK) return rc; }
    const size_t n = (size_t)s->g.nx * s->g.ny * s->g.nz;
    for (int c = 0; c < 5; ++c) {
        int rc = field_out(s, s->r[c], r + c * n, IGR_STORE_F32);
        if (rc != IGR_OK) return rc;
    }
    return igr_sync(s);
}

int igr_get_padded(igr_solver *s, int c, float *f)
{
    if (!s || !f || c < 0 || c > s->nf) return IGR_ERR_ARG;
    if (s->storage == IGR_STORE_F64) return s->fail(IGR_ERR_ARG, "igr_get_padded: not available in the fp64 mode");
    const Grid &g = s->g;
    const void *field = c < s->nf ? s->st[s->cur].f[c] : s->sig[s->sig_cur];
    const size_t wx = g.nx + 2 * IGR_NG, wy = g.ny + 2 * IGR_NG, wz = g.nz + 2 * IGR_NG;
    if (is_device_pointer(f)) {
        launch_pack_padded(g, s->storage, field, f, 0, (int)wz, s->stream);
        return igr_sync(s);
    }
    const size_t plane = wx * wy * 4;
    int chunk = (int)(kStageBytes / plane);
    if (chunk < 1) return s->fail(IGR_ERR_ARG, "igr_get_padded: plane exceeds the staging buffer");
    for (int k0 = 0; k0 < (int)wz; k0 += chunk) {
        const int nk = ((int)wz - k0 < chunk) ? (int)wz - k0 : chunk;
        launch_pack_padded(g, s->storage, field, s->stage, k0, nk, s->stream);
        IGR_CUDA_OK(cudaMemcpyAsync(f + (size_t)k0 * wx * wy, s->stage, nk * plane,
                                    cudaMemcpyDeviceToHost, s->stream));
        IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    }
    return finish(s, "igr_get_padded");
}

// ------------------------------------------------------------------------- rows of the hot path
int igr_halo_bc(igr_solver *s)
{
    if (!s) return IGR_ERR_ARG;
    RowTimer t(s, 0, 1);
    if (s->storage == IGR_STORE_F64) launch64_halo_q(s->g, s->st[s->cur], s->bc64, s->stream);
    else launch_halo_q(s->g, s->storage, s->st[s->cur], s->bc, s->nf, s->stream);
    return finish(s, "igr_halo_bc");
}

int igr_sigma_source(igr_solver *s)
{
    if (!s) return IGR_ERR_ARG;
    RowTimer t(s, 1, s->nf == 7 ? 2 : 1);
    if (s->storage == IGR_STORE_F64) {
        launch64_source(s->g, s->st[s->cur], (double *)s->b, s->alpha, 1.0 / (2.0 * s->dx), s->stream);
        return finish(s, "igr_sigma_source");
    }
    const bool viscous = s->mu > 0 || s->zeta > 0;
    StagePtrs q = s->st[s->cur];
    if (s->nf == 7) {
        // two fluids: the mixture density of every padded cell first; the source kernel then sees
        // (rho, m_x, m_y, m_z) as with one fluid
        launch_rho_total(s->g, (const float *)q.f[0], (const float *)q.f[1], s->rhot, s->stream);
        q.f[0] = s->rhot; q.f[1] = s->st[s->cur].f[2]; q.f[2] = s->st[s->cur].f[3]; q.f[3] = s->st[s->cur].f[4];
    }
    static int no_tma = -1;                  // IGR_SOURCE_TMA=0: the per-thread-load kernel (tuning)
    if (no_tma < 0) { const char *e = getenv("IGR_SOURCE_TMA"); no_tma = (e && atoi(e) == 0) ? 1 : 0; }
    if (s->variant == IGR_VARIANT_TILED && !viscous && !no_tma && s->smaps[s->cur].valid)
        launch_source_tma(s->g, s->storage, s->smaps[s->cur], s->b, (float)s->alpha, (float)(1.0 / (2.0 * s->dx)), s->stream);
    else
        launch_source(s->g, s->storage, q, s->b, (float)s->alpha, (float)(1.0 / (2.0 * s->dx)),
                      viscous ? s->tau : nullptr, (float)s->mu, (float)s->zeta, s->stream);
    return finish(s, "igr_sigma_source");
}

int igr_jacobi(igr_solver *s)
{
    if (!s) return IGR_ERR_ARG;
    const float k2 = (float)(s->alpha / (s->dx * s->dx));
    if (s->storage == IGR_STORE_F64) {
        RowTimer t(s, 2, s->n_jacobi + 1);
        for (int it = 0; it < s->n_jacobi; ++it) {
            launch64_jacobi_sweep(s->g, (const double *)s->st[s->cur].f[0], (const double *)s->b,
                                  (const double *)s->sig[s->sig_cur], (double *)s->sig[1 - s->sig_cur],
                                  s->alpha / (s->dx * s->dx), s->stream);
            s->sig_cur = 1 - s->sig_cur;
        }
        launch64_halo_sigma(s->g, (double *)s->sig[s->sig_cur], s->stream);
        return finish(s, "igr_jacobi");
    }
    if (s->variant == IGR_VARIANT_TILED) {
        // temporally blocked: passes of up to 5 sweeps, each ONE read of rho, b, Sigma and one write
        static int maxns = -1;                   // IGR_JACOBI_MAXNS=1..5: sweeps per blocked pass (tuning)
        if (maxns < 0) { const char *e = getenv("IGR_JACOBI_MAXNS"); maxns = e ? atoi(e) : 5; if (maxns < 1 || maxns > 5) maxns = 5; }
        static int no_tma = -1;                  // IGR_JACOBI_TMA=0: cp.async staging everywhere (tuning)
        if (no_tma < 0) { const char *e = getenv("IGR_JACOBI_TMA"); no_tma = (e && atoi(e) == 0) ? 1 : 0; }
        static int no_quad = -1;                 // IGR_JACOBI_QUAD=0: the blocked kernel in every region (tuning)
        if (no_quad < 0) { const char *e = getenv("IGR_JACOBI_QUAD"); no_quad = (e && atoi(e) == 0) ? 1 : 0; }
        const int npass = (s->n_jacobi + maxns - 1) / maxns;
        RowTimer t(s, 2, 2 * npass + 1);
        for (int left = s->n_jacobi; left > 0; left -= maxns) {
            const bool tma = s->jmaps.valid && !no_tma;
            const int ns = left < maxns ? left : maxns;
            // regions that need no periodic wrap in x / y: four columns per thread (igr_jacobi_quad.cu);
            // the blocked kernel keeps the others
            JacobiQuadPlan quad = {};
            if (tma && !no_quad) quad = jacobi_quad_plan(s->g, ns, k2);
            launch_jacobi_blocked(s->g, s->storage, ns, s->nf == 7 ? (void *)s->rhot : s->st[s->cur].f[0], s->b,
                                  s->sig[s->sig_cur], s->sig[1 - s->sig_cur], k2,
                                  tma ? &s->jmaps.rho[s->cur] : nullptr, tma ? &s->jmaps.b : nullptr,
                                  tma ? &s->jmaps.sig[s->sig_cur] : nullptr, &quad, s->stream);
            if (quad.nbx > 0) {
                const JacobiMaps &jm = quad.wy ? s->jmaps2 : s->jmaps;
                launch_jacobi_quad(s->g, s->storage, ns, quad, s->sig[1 - s->sig_cur], k2, &jm.rho[s->cur], &jm.b,
                                   &jm.sig[s->sig_cur], s->stream);
            }
            s->sig_cur = 1 - s->sig_cur;
        }
        launch_halo_sigma(s->g, s->storage, s->sig[s->sig_cur], s->stream);
        return finish(s, "igr_jacobi");
    }
    RowTimer t(s, 2, s->n_jacobi + 1);
    for (int it = 0; it < s->n_jacobi; ++it) {
        launch_jacobi_sweep(s->g, s->storage, s->nf == 7 ? (void *)s->rhot : s->st[s->cur].f[0], s->b, s->sig[s->sig_cur],
                            s->sig[1 - s->sig_cur], k2, s->stream);
        s->sig_cur = 1 - s->sig_cur;
    }
    launch_halo_sigma(s->g, s->storage, s->sig[s->sig_cur], s->stream);
    return finish(s, "igr_jacobi");
}

int igr_rhs(igr_solver *s)
{
    if (!s) return IGR_ERR_ARG;
    if (s->nf != 5) return s->fail(IGR_ERR_ARG, "two fluids: only the fused step (igr_step / igr_stage) is built");
    { const int rc = ensure_r(s); if (rc != IGR_OK) return rc; }
    RowTimer t(s, 3, 1);
    if (s->storage == IGR_STORE_F64) {
        double *r64[5];
        for (int c = 0; c < 5; ++c) r64[c] = (double *)s->r[c];
        launch64_rhs(s->g, s->order, s->st[s->cur], (const double *)s->sig[s->sig_cur], r64, s->gamma, s->dx, s->stream);
        return finish(s, "igr_rhs");
    }
    RhsParams p;
    p.gamma = (float)s->gamma; p.inv_dx = (float)(1.0 / s->dx); p.order = s->order;
    if (s->variant == IGR_VARIANT_TILED) {
        RhsTileArgs a = {};
        for (int c = 0; c < 5; ++c) a.r[c] = s->r[c];
        a.gamma = p.gamma; a.inv_dx = p.inv_dx; a.zc = 0;
        launch_rhs_tile(s->g, s->storage, s->order, false, s->maps.q[s->cur], s->maps.sig[s->sig_cur], a, s->stream);
    } else {
        launch_rhs_simple(s->g, s->storage, s->st[s->cur], s->sig[s->sig_cur], s->r, p, s->stream);
    }
    if (s->mu > 0 || s->zeta > 0) {
        // viscous fluxes: ghosts of the stress fields by the BC index map, then r += -div F_visc
        launch_halo_fields(s->g, s->tau, 6, s->stream);
        if (s->variant == IGR_VARIANT_TILED) {
            ViscTileArgs a = {};
            for (int c = 0; c < 5; ++c) { a.q[c] = s->st[s->cur].f[c]; a.r[c] = s->r[c]; }
            a.tau = s->tau; a.inv_dx = p.inv_dx; a.zc = 0;
            launch_viscous_tile(s->g, s->storage, s->order, false, s->vmaps.q[s->cur], s->vmaps.tau, a, s->stream);
        } else {
            launch_viscous_add(s->g, s->storage, s->order, s->st[s->cur], s->tau, s->r, p.inv_dx, s->stream);
        }
        s->launches += 2;
    }
    return finish(s, "igr_rhs");
}

// Unfused buffer discipline (only the current sub-step enters the RHS; the buffer
// with q^n is only read by the update): A = st[0] holds q^n, B = st[1] the sub-step.
//   stage 1: B = A + dt r(A);  stage 2: B = A + 1/4((B - A) + dt r(B));  stage 3: A = A + 2/3((B - A) + dt r(B))
int igr_rk_update(igr_solver *s, int stage, double dt)
{
    if (!s || stage < 1 || stage > 3) return IGR_ERR_ARG;
    if (s->nf != 5) return s->fail(IGR_ERR_ARG, "two fluids: only the fused step (igr_step / igr_stage) is built");
    { const int rc = ensure_r(s); if (rc != IGR_OK) return rc; }
    const float beta = stage == 1 ? 1.0f : (stage == 2 ? 0.25f : (float)(2.0 / 3.0));
    StagePtrs &A = s->st[0], &B = s->st[1];
    RowTimer t(s, 4, 1);
    if (s->storage == IGR_STORE_F64) {
        double *r64[5];
        for (int c = 0; c < 5; ++c) r64[c] = (double *)s->r[c];
        const double b64 = stage == 1 ? 1.0 : (stage == 2 ? 0.25 : 2.0 / 3.0);
        if (stage == 3) IGR_CUDA_OK(cudaMemsetAsync(s->wave, 0, sizeof(WaveResult64), s->stream));
        launch64_rk_update(s->g, A, stage == 1 ? A : B, stage == 3 ? A : B, r64, b64, dt, s->gamma,
                           stage == 3 ? (WaveResult64 *)s->wave : nullptr, s->stream);
        s->cur = stage == 3 ? 0 : 1;
        s->wave_valid = stage == 3;
        return finish(s, "igr_rk_update");
    }
    if (stage == 1) {
        launch_rk_update(s->g, s->storage, A, A, B, s->r, beta, (float)dt, (float)s->gamma, nullptr, s->stream);
        s->cur = 1;
        s->wave_valid = false;                   // the cached speed is the one of q^n, not of this sub-step
    } else if (stage == 2) {
        launch_rk_update(s->g, s->storage, A, B, B, s->r, beta, (float)dt, (float)s->gamma, nullptr, s->stream);
        s->cur = 1;
        s->wave_valid = false;
    } else {
        IGR_CUDA_OK(cudaMemsetAsync(s->wave, 0, sizeof(WaveResult), s->stream));
        launch_rk_update(s->g, s->storage, A, B, A, s->r, beta, (float)dt, (float)s->gamma, s->wave, s->stream);
        s->cur = 0;
        s->wave_valid = true;
    }
    return finish(s, "igr_rk_update");
}

int igr_stage(igr_solver *s, int stage, double dt)
{
    if (!s || stage < 1 || stage > 3) return IGR_ERR_ARG;
    {
        const int fused3 = (s->fused && s->variant == IGR_VARIANT_TILED) ? 2 : 1;
        const int want = stage == 1 ? 0 : (stage == 2 ? 1 : fused3);
        if (s->cur != want) return s->fail(IGR_ERR_ARG, "igr_stage: stages must run in the order 1, 2, 3");
    }
    {
        int rc;
        if ((rc = igr_halo_bc(s)) != IGR_OK) return rc;
        if ((rc = igr_sigma_source(s)) != IGR_OK) return rc;
        if ((rc = igr_jacobi(s)) != IGR_OK) return rc;
        const bool viscous = s->mu > 0 || s->zeta > 0;
        if (s->fused && s->variant == IGR_VARIANT_TILED) {
            // RHS + stage update + (stage 3) wave speed in one kernel: q^n = st[0] is only read
            // pointwise, the sub-steps alternate st[1], st[2]; stage 3 writes st[0] in place.
            // With viscosity the inviscid RHS kernel stores r and the viscous kernel carries the update.
            RowTimer t(s, 3, viscous ? 3 : 1);
            const int src = s->cur, dst = stage == 1 ? 1 : (stage == 2 ? 2 : 0);
            const float beta = stage == 1 ? 1.0f : (stage == 2 ? 0.25f : (float)(2.0 / 3.0));
            if (stage == 3) IGR_CUDA_OK(cudaMemsetAsync(s->wave, 0, sizeof(WaveResult), s->stream));
            RhsTileArgs a = {};
            a.gamma = (float)s->gamma; a.inv_dx = (float)(1.0 / s->dx); a.zc = 0;
            a.nf = s->nf;
            if (s->nf == 7) { a.k1 = (float)(1.0 / (s->gamma - 1.0)); a.k2 = (float)(1.0 / (s->gamma2 - 1.0)); }
            if (!viscous) {
                for (int c = 0; c < s->nf; ++c) { a.qn[c] = s->st[0].f[c]; a.qout[c] = s->st[dst].f[c]; }
                a.beta = beta; a.dt = (float)dt; a.read_qn = stage != 1;
                if (stage == 3) a.wave = s->wave;
                launch_rhs_tile(s->g, s->storage, s->order, true, s->maps.q[src], s->maps.sig[s->sig_cur], a, s->stream);
            } else {
                if ((rc = ensure_r(s)) != IGR_OK) return rc;
                for (int c = 0; c < 5; ++c) a.r[c] = s->r[c];
                launch_rhs_tile(s->g, s->storage, s->order, false, s->maps.q[src], s->maps.sig[s->sig_cur], a, s->stream);
                launch_halo_fields(s->g, s->tau, 6, s->stream);
                ViscTileArgs v = {};
                for (int c = 0; c < 5; ++c) {
                    v.q[c] = s->st[src].f[c]; v.r[c] = s->r[c]; v.qn[c] = s->st[0].f[c]; v.qout[c] = s->st[dst].f[c];
                }
                v.tau = s->tau; v.inv_dx = a.inv_dx; v.zc = 0;
                v.beta = beta; v.dt = (float)dt; v.gamma = a.gamma; v.read_qn = stage != 1;
                if (stage == 3) v.wave = s->wave;
                launch_viscous_tile(s->g, s->storage, s->order, true, s->vmaps.q[src], s->vmaps.tau, v, s->stream);
            }
            s->cur = dst;
            s->wave_valid = stage == 3;          // the cached speed belongs to q^n / q^{n+1} only
            if ((rc = finish(s, "igr_step (fused rhs)")) != IGR_OK) return rc;
        } else {
            if ((rc = igr_rhs(s)) != IGR_OK) return rc;
            if ((rc = igr_rk_update(s, stage, dt)) != IGR_OK) return rc;
        }
    }
    return IGR_OK;
}

int igr_step(igr_solver *s, double dt)
{
    if (!s) return IGR_ERR_ARG;
    if (s->cur != 0) return s->fail(IGR_ERR_ARG, "igr_step: called in the middle of a step");
    for (int stage = 1; stage <= 3; ++stage) {
        const int rc = igr_stage(s, stage, dt);
        if (rc != IGR_OK) return rc;
    }
    return IGR_OK;
}

// ------------------------------------------------------------------------- NEXT-2: slab exchange
// z is the slowest axis of the padded layout: a range of planes of one field is one contiguous chunk.
int igr_export_fields(igr_solver *s, igr_export *out)
{
    if (!s || !out) return IGR_ERR_ARG;
    if (s->nf != 5) return s->fail(IGR_ERR_ARG, "two fluids: the slab exchange is not built");
    if (s->storage == IGR_STORE_F64) return s->fail(IGR_ERR_ARG, "fp64 mode: the slab exchange is not built");
    memset(out, 0, sizeof *out);
    out->base = (uint64_t)(uintptr_t)s->base;
    for (int b = 0; b < 3; ++b)
        for (int c = 0; c < 5; ++c) out->q_offset[b][c] = (uint64_t)((char *)s->st[b].f[c] - s->base);
    for (int b = 0; b < 2; ++b) out->sig_offset[b] = (uint64_t)((char *)s->sig[b] - s->base);
    out->plane_bytes = (uint64_t)s->g.sz * (s->storage == IGR_STORE_F32 ? 4 : 2);
    out->nz = s->g.nz; out->storage = s->storage;
    out->cur = s->cur; out->sig_cur = s->sig_cur;
    out->owns_memory = s->owns_base ? 1 : 0;
    if (s->owns_base) {
        cudaIpcMemHandle_t h;
        static_assert(sizeof h == sizeof out->ipc_handle, "igr_export.ipc_handle must hold a cudaIpcMemHandle_t");
        IGR_CUDA_OK(cudaIpcGetMemHandle(&h, s->base));
        memcpy(out->ipc_handle, &h, sizeof h);
    }
    return IGR_OK;
}

int igr_ipc_open(const igr_export *peer, void **peer_base)
{
    if (!peer || !peer_base || !peer->owns_memory) return IGR_ERR_ARG;
    cudaIpcMemHandle_t h;
    memcpy(&h, peer->ipc_handle, sizeof h);
    *peer_base = nullptr;
    if (cudaIpcOpenMemHandle(peer_base, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) {
        cudaGetLastError();
        return IGR_ERR_CUDA;
    }
    return IGR_OK;
}

int igr_ipc_close(void *peer_base)
{
    if (!peer_base) return IGR_ERR_ARG;
    if (cudaIpcCloseMemHandle(peer_base) != cudaSuccess) { cudaGetLastError(); return IGR_ERR_CUDA; }
    return IGR_OK;
}

int igr_set_neighbor(igr_solver *s, int side, const igr_export *peer, const void *peer_base, int dst_plane,
                     int src_plane, int count)
{
    if (!s || side < 0 || side > 1) return IGR_ERR_ARG;
    igr_solver::Neighbor &nb = s->nb[side];
    if (!peer) { nb.active = false; return IGR_OK; }            // unregister
    if (!peer_base || count < 1) return IGR_ERR_ARG;
    if (s->g.bc[4 + side] != kBcExternal)
        return s->fail(IGR_ERR_BC, "igr_set_neighbor: that z face is not IGR_BC_EXTERNAL");
    const uint64_t pb = (uint64_t)s->g.sz * (s->storage == IGR_STORE_F32 ? 4 : 2);
    if (peer->plane_bytes != pb || peer->storage != s->storage)
        return s->fail(IGR_ERR_ARG, "igr_set_neighbor: the neighbour's planes have another shape or element type");
    if (dst_plane < -IGR_NG || dst_plane + count > s->g.nz + IGR_NG || src_plane < 0 || src_plane + count > peer->nz)
        return s->fail(IGR_ERR_ARG, "igr_set_neighbor: plane range outside the padded array / the neighbour's interior");
    nb.active = true; nb.desc = *peer; nb.base = (const char *)peer_base;
    nb.dst = dst_plane; nb.src = src_plane; nb.count = count;
    return IGR_OK;
}

int igr_pull_halo(igr_solver *s)
{
    if (!s) return IGR_ERR_ARG;
    const size_t pb = (size_t)s->g.sz * (s->storage == IGR_STORE_F32 ? 4 : 2);
    for (int side = 0; side < 2; ++side) {
        const igr_solver::Neighbor &nb = s->nb[side];
        if (!nb.active) continue;
        const size_t doff = (size_t)(nb.dst + IGR_NG) * pb, soff = (size_t)(nb.src + IGR_NG) * pb, n = (size_t)nb.count * pb;
        for (int c = 0; c < 5; ++c)
            IGR_CUDA_OK(cudaMemcpyAsync((char *)s->st[s->cur].f[c] + doff, nb.base + nb.desc.q_offset[s->cur][c] + soff, n,
                                        cudaMemcpyDeviceToDevice, s->stream));
        IGR_CUDA_OK(cudaMemcpyAsync((char *)s->sig[s->sig_cur] + doff, nb.base + nb.desc.sig_offset[s->sig_cur] + soff, n,
                                    cudaMemcpyDeviceToDevice, s->stream));
    }
    // the cached wave speed stays valid if no plane that entered it was overwritten (igr_set_wave_range)
    for (int side = 0; side < 2; ++side) {
        const igr_solver::Neighbor &nb = s->nb[side];
        if (nb.active && nb.dst < s->g.wk1 && nb.dst + nb.count > s->g.wk0) s->wave_valid = false;
    }
    return IGR_OK;
}

// ---- interprocess events (igr.h): stream-ordered ordering of the exchange
static int ensure_event(igr_solver *s, int which)
{
    if (s->ipc_ev[which]) return IGR_OK;
    IGR_CUDA_OK(cudaEventCreateWithFlags(&s->ipc_ev[which], cudaEventDisableTiming | cudaEventInterprocess));
    // an event that was never recorded counts as complete; record it once so that a neighbour that opens the
    // handle before the first stage waits on something well defined
    IGR_CUDA_OK(cudaEventRecord(s->ipc_ev[which], s->stream));
    return IGR_OK;
}

int igr_event_handle(igr_solver *s, int which, unsigned char handle[64])
{
    if (!s || !handle || which < 0 || which > 1) return IGR_ERR_ARG;
    { const int rc = ensure_event(s, which); if (rc != IGR_OK) return rc; }
    cudaIpcEventHandle_t h;
    static_assert(sizeof h == 64, "cudaIpcEventHandle_t is 64 bytes");
    IGR_CUDA_OK(cudaIpcGetEventHandle(&h, s->ipc_ev[which]));
    memcpy(handle, &h, sizeof h);
    return IGR_OK;
}

int igr_event_open(const unsigned char handle[64], void **event)
{
    if (!handle || !event) return IGR_ERR_ARG;
    cudaIpcEventHandle_t h;
    memcpy(&h, handle, sizeof h);
    cudaEvent_t e = nullptr;
    if (cudaIpcOpenEventHandle(&e, h) != cudaSuccess) { cudaGetLastError(); *event = nullptr; return IGR_ERR_CUDA; }
    *event = (void *)e;
    return IGR_OK;
}

int igr_event_close(void *event)
{
    if (!event) return IGR_ERR_ARG;
    if (cudaEventDestroy((cudaEvent_t)event) != cudaSuccess) { cudaGetLastError(); return IGR_ERR_CUDA; }
    return IGR_OK;
}

int igr_event_record(igr_solver *s, int which)
{
    if (!s || which < 0 || which > 1) return IGR_ERR_ARG;
    { const int rc = ensure_event(s, which); if (rc != IGR_OK) return rc; }
    IGR_CUDA_OK(cudaEventRecord(s->ipc_ev[which], s->stream));
    return IGR_OK;
}

int igr_event_wait(igr_solver *s, void *event)
{
    if (!s || !event) return IGR_ERR_ARG;
    IGR_CUDA_OK(cudaStreamWaitEvent(s->stream, (cudaEvent_t)event, 0));
    return IGR_OK;
}

int igr_set_wave_range(igr_solver *s, int k0, int k1)
{
    if (!s || k0 < 0 || k1 > s->g.nz || k0 >= k1) return IGR_ERR_ARG;
    s->g.wk0 = k0; s->g.wk1 = k1;
    s->wave_valid = false;
    return IGR_OK;
}

int igr_max_wavespeed(igr_solver *s, double *out)
{
    if (!s || !out) return IGR_ERR_ARG;
    if (s->storage == IGR_STORE_F64) {
        if (!s->wave_valid) {
            RowTimer t(s, 5, 1);
            IGR_CUDA_OK(cudaMemsetAsync(s->wave, 0, sizeof(WaveResult64), s->stream));
            launch64_wavespeed(s->g, s->st[s->cur], s->gamma, (WaveResult64 *)s->wave, s->stream);
            s->wave_valid = (s->cur == 0);
        }
        WaveResult64 h;
        IGR_CUDA_OK(cudaMemcpyAsync(&h, s->wave, sizeof h, cudaMemcpyDeviceToHost, s->stream));
        IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
        int rc = finish(s, "igr_max_wavespeed");
        if (rc != IGR_OK) return rc;
        double v;
        memcpy(&v, &h.max_bits, 8);
        *out = v;
        if (h.nonfinite || !(v > 0.0) || !std::isfinite(v))
            return s->fail(IGR_ERR_NONFINITE, "igr_max_wavespeed: non-finite state (NaN/Inf, or negative pressure/density)");
        return IGR_OK;
    }
    if (!s->wave_valid) {
        RowTimer t(s, 5, 1);
        IGR_CUDA_OK(cudaMemsetAsync(s->wave, 0, sizeof(WaveResult), s->stream));
        if (s->nf == 7)
            launch_wavespeed2(s->g, s->st[s->cur], (float)(1.0 / (s->gamma - 1.0)), (float)(1.0 / (s->gamma2 - 1.0)),
                              s->wave, s->stream);
        else
            launch_wavespeed(s->g, s->storage, s->st[s->cur], (float)s->gamma, s->wave, s->stream);
        s->wave_valid = (s->cur == 0);
    }
    WaveResult h;
    IGR_CUDA_OK(cudaMemcpyAsync(&h, s->wave, sizeof h, cudaMemcpyDeviceToHost, s->stream));
    IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    int rc = finish(s, "igr_max_wavespeed");
    if (rc != IGR_OK) return rc;
    float v;
    memcpy(&v, &h.max_bits, 4);
    *out = (double)v;
    if (h.nonfinite || !(v > 0.0f) || !std::isfinite(v))
        return s->fail(IGR_ERR_NONFINITE, "igr_max_wavespeed: non-finite state (NaN/Inf, or negative pressure/density)");
    return IGR_OK;
}

int igr_set_viscosity(igr_solver *s, double mu, double zeta)
{
    if (!s || !(mu >= 0) || !(zeta >= 0)) return IGR_ERR_ARG;
    if (s->nf != 5 && (mu > 0 || zeta > 0)) return s->fail(IGR_ERR_ARG, "two fluids: viscous fluxes are not built");
    if (s->storage == IGR_STORE_F64 && (mu > 0 || zeta > 0)) return s->fail(IGR_ERR_ARG, "fp64 mode: viscous fluxes are not built");
    if ((mu > 0 || zeta > 0) && !s->tau) {
        if (cudaMalloc((void **)&s->tau, (size_t)s->g.np * 6 * 4) != cudaSuccess) {
            cudaGetLastError();
            s->tau = nullptr;
            return s->fail(IGR_ERR_ALLOC, "igr_set_viscosity: cudaMalloc of the stress fields failed");
        }
        IGR_CUDA_OK(cudaMemsetAsync(s->tau, 0, (size_t)s->g.np * 6 * 4, s->stream));
        if (s->variant == IGR_VARIANT_TILED) {
            const char *msg = "";
            if (visc_tile_make_maps(s->g, s->storage, s->st, 3, s->tau, &s->vmaps, &msg) != 0) {
                cudaFree(s->tau);                // a later call must not find stress fields without maps
                s->tau = nullptr;
                return s->fail(IGR_ERR_CUDA, msg);
            }
        }
    }
    s->mu = mu; s->zeta = zeta;
    return IGR_OK;
}

int igr_kernel_launches(igr_solver *s, long long *out)
{
    if (!s || !out) return IGR_ERR_ARG;
    *out = s->launches;
    return IGR_OK;
}

int igr_profile(igr_solver *s, int enable)
{
    if (!s) return IGR_ERR_ARG;
    IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    for (cudaEvent_t e : s->ev) cudaEventDestroy(e);
    s->ev.clear(); s->ev_row.clear();
    s->profile = enable != 0;
    return IGR_OK;
}

int igr_profile_read(igr_solver *s, double ms[6], long long count[6])
{
    if (!s || !ms || !count) return IGR_ERR_ARG;
    IGR_CUDA_OK(cudaStreamSynchronize(s->stream));
    for (int r = 0; r < 6; ++r) { ms[r] = 0.0; count[r] = 0; }
    for (size_t i = 0; i < s->ev_row.size(); ++i) {
        float t = 0.f;
        IGR_CUDA_OK(cudaEventElapsedTime(&t, s->ev[2 * i], s->ev[2 * i + 1]));
        ms[s->ev_row[i]] += t; count[s->ev_row[i]] += 1;
    }
    return IGR_OK;
}

}  // extern "C"
