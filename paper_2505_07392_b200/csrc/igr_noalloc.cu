// igr_noalloc.cu -- igr_max_wavespeed_noalloc: row a6 (the CFL wave speed, Alg. 1; DESIGN.md
// readings A5/A9) for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc.  The entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//
// A variant of k_wavespeed (igr_kernels.cu).  That kernel reduces into a WaveResult accumulator which igr_create
// allocates; this one needs no solver and no allocation: every block writes its partial maximum into a FILE-SCOPE
// device array (the scratch), a second one-block kernel reduces the partials into the caller's output.  The
// per-cell arithmetic is the same inline function (wavespeed_of, igr_common.cuh), and a maximum does not depend on
// the order of its operands, so the result is bitwise that of igr_max_wavespeed on an fp32-stored state.
//
// The scratch: IGR_NOALLOC_MAX_BLOCKS partials of 8 bytes = 512 KB, held by every GPU that loads the library until the
// process exits.  One block takes 16384 cells, so the largest state is IGR_NOALLOC_MAX_CELLS = 2^30 cells (1024^3);
// larger ones are refused.  EVERY call on a device shares the array: two calls that overlap on the GPU (different
// streams, or two host threads) race on it -- callers order them on one stream.  The array keeps the last call's
// contents; nothing in it has to start at zero, because the first kernel overwrites every slot the second one reads
// (slots [0, blocks of THIS call)), so no clearing pass is needed and stale slots beyond that range are never read.
//
// In host code the array's name is a host-side stand-in, not a device address.  The address comes from
// cudaGetSymbolAddress, once per device, with that device current (first call on the device; checked).
#include "igr_common.cuh"
#include "../../include/igr.h"

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_PER_THREAD = 64;
constexpr int NA_CELLS_PER_BLOCK = NA_THREADS * NA_PER_THREAD;          // 16384
constexpr int NA_MAX_BLOCKS = 65536;
constexpr int NA_MAX_DEVICES = 64;
static_assert((long long)NA_CELLS_PER_BLOCK * NA_MAX_BLOCKS == IGR_NOALLOC_MAX_CELLS, "igr.h states the limit");

struct NaPartial {
    float vmax;               // partial maximum of max_d |u_d| + c
    unsigned int bad;         // != 0: a cell of the block gave a non-finite value
};

static __device__ __align__(256) NaPartial g_noalloc_scratch[NA_MAX_BLOCKS];   // 512 KB per GPU, until exit

// pass 1: block b takes cells [b * 16384, (b + 1) * 16384) of the unpadded fields q[c][cell], c = 0..4
__global__ void __launch_bounds__(NA_THREADS)
k_wavespeed_partials(const float *__restrict__ q, long long n, float gamma, NaPartial *__restrict__ part)
{
    __shared__ float s_v[NA_THREADS / 32];
    __shared__ unsigned int s_b[NA_THREADS / 32];
    const long long base = (long long)blockIdx.x * NA_CELLS_PER_BLOCK;
    float vmax = 0.f;
    bool bad = false;
#pragma unroll 4
    for (int it = 0; it < NA_PER_THREAD; ++it) {
        const long long t = base + (long long)it * NA_THREADS + threadIdx.x;
        if (t < n)
            vmax = fmaxf(vmax, wavespeed_of(q[t], q[n + t], q[2 * n + t], q[3 * n + t], q[4 * n + t], gamma, bad));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    const bool anybad = __any_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = vmax; s_b[threadIdx.x >> 5] = anybad ? 1u : 0u; }
    __syncthreads();
    if (threadIdx.x == 0) {
        NaPartial p = { 0.f, 0u };
#pragma unroll
        for (int w = 0; w < NA_THREADS / 32; ++w) { p.vmax = fmaxf(p.vmax, s_v[w]); p.bad |= s_b[w]; }
        part[blockIdx.x] = p;
    }
}

// pass 2: one block reduces the nb partials of THIS call into out[0] = maximum, out[1] = 1 if non-finite else 0
__global__ void __launch_bounds__(1024) k_wavespeed_final(const NaPartial *__restrict__ part, int nb, float *out)
{
    __shared__ float s_v[32];
    __shared__ unsigned int s_b[32];
    float vmax = 0.f;
    unsigned int bad = 0u;
    for (int b = threadIdx.x; b < nb; b += blockDim.x) { vmax = fmaxf(vmax, part[b].vmax); bad |= part[b].bad; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    const bool anybad = __any_sync(0xffffffffu, bad != 0u);
    if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = vmax; s_b[threadIdx.x >> 5] = anybad ? 1u : 0u; }
    __syncthreads();
    if (threadIdx.x == 0) {
        float v = 0.f;
        unsigned int f = 0u;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { v = fmaxf(v, s_v[w]); f |= s_b[w]; }
        out[0] = v;
        out[1] = f ? 1.0f : 0.0f;
    }
}

// the message goes into the caller's buffer (vsnprintf: no allocation)
__attribute__((format(printf, 4, 5))) int na_fail(int code, char *errbuf, size_t len, const char *fmt, ...)
{
    if (errbuf && len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(errbuf, len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// device address of the scratch on the CURRENT device (resolved once per device; no allocation)
int na_scratch(NaPartial **out, char *errbuf, size_t len)
{
    static std::mutex mu;
    static NaPartial *addr[NA_MAX_DEVICES] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess)
        return na_fail(IGR_ERR_CUDA, errbuf, len, "igr_max_wavespeed_noalloc: cudaGetDevice failed: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES)
        return na_fail(IGR_ERR_ARG, errbuf, len, "igr_max_wavespeed_noalloc: device %d is beyond the %d devices served", dev,
                       NA_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        NaPartial *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p)
            return na_fail(IGR_ERR_CUDA, errbuf, len,
                           "igr_max_wavespeed_noalloc: cudaGetSymbolAddress of the scratch failed on device %d (%d): %s", dev,
                           (int)e, cudaGetErrorString(e));
        addr[dev] = p;
    }
    *out = addr[dev];
    return IGR_OK;
}

}  // namespace

extern "C" int igr_max_wavespeed_noalloc(const float *q, int nx, int ny, int nz, double gamma, float *out,
                                         void *stream, char *errbuf, size_t errbuf_len)
{
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (!q || !out) return na_fail(IGR_ERR_ARG, errbuf, errbuf_len, "igr_max_wavespeed_noalloc: null pointer");
    if (nx <= 0 || ny <= 0 || nz <= 0 || !(gamma > 1.0))
        return na_fail(IGR_ERR_ARG, errbuf, errbuf_len,
                       "igr_max_wavespeed_noalloc: sizes must be positive and gamma > 1 (got %d x %d x %d, gamma %g)", nx, ny, nz,
                       gamma);
    const long long n = (long long)nx * ny * nz;
    if (n > IGR_NOALLOC_MAX_CELLS)
        return na_fail(IGR_ERR_ARG, errbuf, errbuf_len,
                       "igr_max_wavespeed_noalloc: %lld cells exceed the static scratch (IGR_NOALLOC_MAX_CELLS = %lld)", n,
                       (long long)IGR_NOALLOC_MAX_CELLS);
    NaPartial *part = nullptr;
    const int rc = na_scratch(&part, errbuf, errbuf_len);
    if (rc != IGR_OK) return rc;
    const int nb = (int)((n + NA_CELLS_PER_BLOCK - 1) / NA_CELLS_PER_BLOCK);
    cudaStream_t st = (cudaStream_t)stream;
    k_wavespeed_partials<<<nb, NA_THREADS, 0, st>>>(q, n, (float)gamma, part);
    k_wavespeed_final<<<1, 1024, 0, st>>>(part, nb, out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess)
        return na_fail(IGR_ERR_CUDA, errbuf, errbuf_len, "igr_max_wavespeed_noalloc: launch failed: %s", cudaGetErrorString(e));
    return IGR_OK;
}
