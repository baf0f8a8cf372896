// igr_tma.cuh -- the few sm_100a primitives the streaming kernels share: mbarrier (init / expect_tx / parity wait),
// tiled TMA loads (cp.async.bulk.tensor, 3-D and 4-D boxes) and the host-side tensor-map encoder.
//
// Rules these kernels rely on (B200, measured): the shared-memory destination of a box is 128-byte aligned; the
// box's innermost start coordinate must land on a 16-byte boundary of the row (otherwise the load raises "illegal
// instruction"), so boxes start at a column rounded down to 16 bytes; global strides are multiples of 16 bytes
// (the padded layout of igr_common.cuh guarantees it); a slot read through the generic proxy is handed back to
// the async proxy with fence.proxy.async before it is refilled.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace igr_tma {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
// after the mbarrier.init of one thread and before the first TMA issue
__device__ __forceinline__ void fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// generic-proxy reads of a slot are done (barrier since): make it writable by the async proxy again
__device__ __forceinline__ void fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// spin on the phase parity; `bar` is a shared-window address (smem_u32)
__device__ __forceinline__ void mbar_wait_s32(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "IGR_MBAR_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra IGR_MBAR_DONE;\n"
        "bra IGR_MBAR_WAIT;\n"
        "IGR_MBAR_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) { mbar_wait_s32(smem_u32(bar), parity); }

__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, int c3, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

// ---- host: cuTensorMapEncodeTiled through the runtime's driver entry point (libigr does not link libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

inline EncodeTiledFn get_encode()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

inline CUtensorMapDataType data_type(int storage)      // IGR_STORE_F32 / F16 / BF16
{
    return storage == 0 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                        : (storage == 1 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16);
}

// rank-3 or rank-4 tiled map, no interleave, no swizzle, zero fill outside the tensor
inline bool encode(CUtensorMap *out, CUtensorMapDataType dt, int rank, const void *base, const cuuint64_t *dims,
                   const cuuint64_t *strides, const cuuint32_t *box)
{
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    const cuuint32_t estr[4] = { 1, 1, 1, 1 };
    return enc(out, dt, (cuuint32_t)rank, const_cast<void *>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace igr_tma
