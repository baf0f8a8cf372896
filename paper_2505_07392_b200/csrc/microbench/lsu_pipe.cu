// lsu_pipe.cu -- microbenchmark behind the design of k_jacobi_quad: do SHFL and LDS share a pipe
// on sm_100a, and what do 128-bit shared-memory accesses cost?  Not part of libigr.so.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o lsu_pipe lsu_pipe.cu && ./lsu_pipe
// One CTA of 512 threads per SM; every mode issues the named instructions per unrolled step with addresses that
// change every step (nothing can be hoisted).  Result on B200 (profiles/r02_microbench_lsu.txt): LDS.32 and SHFL cost one
// clock per warp instruction per SM each and ADD (4 + 4 take 8 clocks): one pipe; LDS.128 / STS.128 cost 4 clocks.
#include <cstdio>
#include <cuda_runtime.h>
template <int MODE>
__global__ void __launch_bounds__(512, 1) k(float *out, int iters, int stride)
{
    __shared__ float sm[8192];
    const int t = threadIdx.x;
    for (int i = t; i < 8192; i += 512) sm[i] = i & 3;
    __syncthreads();
    float a0 = t, a1 = t + 1, a2 = t + 2, a3 = t + 3, a4 = 0, a5 = 0, a6 = 0, a7 = 0;
    int off = t;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            off = (off + stride) & 1023;          // address changes every step (not hoistable)
            const float *p = sm + off;
            if (MODE == 0 || MODE == 2 || MODE == 5) {      // 4 LDS.32
                a0 += p[0]; a1 += p[1024]; a2 += p[2048]; a3 += p[3072];
            }
            if (MODE == 2) {                   // 4 SHFL (of values the loads just changed)
                a4 += __shfl_up_sync(0xffffffffu, a0, 1); a5 += __shfl_down_sync(0xffffffffu, a1, 1);
                a6 += __shfl_up_sync(0xffffffffu, a2, 1); a7 += __shfl_down_sync(0xffffffffu, a3, 1);
            }
            if (MODE == 3) {                   // 1 LDS.128 (4 wavefronts)
                float4 v = *reinterpret_cast<const float4 *>(sm + ((off * 4) & 4095)); a0 += v.x; a1 += v.y; a2 += v.z; a3 += v.w;
            }
            if (MODE == 7) {                   // 1 LDS.128 + 1 STS.128
                float4 v = *reinterpret_cast<const float4 *>(sm + ((off * 4) & 4095)); a0 += v.x; a1 += v.y; a2 += v.z; a3 += v.w;
                *reinterpret_cast<float4 *>(sm + 4096 + ((off * 4) & 4095)) = make_float4(a0, a1, a2, a3);
            }
            if (MODE == 4 || MODE == 5) {                   // 16 FFMA
#pragma unroll
                for (int r = 0; r < 2; ++r) {
                    a4 = fmaf(a4, 1.0001f, a0); a5 = fmaf(a5, 1.0001f, a1); a6 = fmaf(a6, 1.0001f, a2); a7 = fmaf(a7, 1.0001f, a3);
                    a4 = fmaf(a4, 1.0002f, a1); a5 = fmaf(a5, 1.0002f, a2); a6 = fmaf(a6, 1.0002f, a3); a7 = fmaf(a7, 1.0002f, a0);
                }
            }
        }
    }
    out[blockIdx.x * 512 + t] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
}
template <int MODE> void run(const char *name, double n_instr, int stride = 32)
{
    float *out; cudaMalloc(&out, 148 * 512 * 4);
    const int iters = 20000;
    k<MODE><<<148, 512>>>(out, 100, stride);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    cudaEventRecord(a);
    k<MODE><<<148, 512>>>(out, iters, stride);
    cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    double cyc = ms * 1e-3 * 1.965e9 / iters / 8.0;      // per unroll step, all 16 warps of the SM
    printf("%-28s %8.3f ms  %7.2f clk per step per SM (16 warps) = %.2f clk per warp-instr\n", name, ms, cyc, cyc / (16 * n_instr));
    cudaFree(out);
}
int main()
{
    run<4>("warm", 16);
    run<0>("4 LDS.32", 4);
    run<2>("4 LDS.32 + 4 SHFL", 8);
    run<3>("1 LDS.128", 1);
    run<7>("1 LDS.128 + 1 STS.128", 2);
    run<4>("16 FFMA", 16);
    run<5>("4 LDS.32 + 16 FFMA", 20);
    return 0;
}
