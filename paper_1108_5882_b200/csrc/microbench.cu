// microbench.cu — register-resident peak probes used as roofline denominators
// (MEASURED_PEAKS.json has no fp64 figure): fp64 FMA, fp64 mma.sync m8n8k4, HBM read stream.
#include "pwa_internal.h"

namespace pwa {

__global__ void __launch_bounds__(256) k_mb_dfma(double *out, int iters, double seed)
{
    double a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = seed + k + threadIdx.x * 1e-3;
    const double x = 1.0000001, y = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] = fma(a[k], x, y);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k];
    if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(256) k_mb_dmma(double *out, int iters, double seed)
{
    double c[8][2];
#pragma unroll
    for (int k = 0; k < 8; ++k) { c[k][0] = seed + k; c[k][1] = seed - k; }
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1e-3 + threadIdx.x * 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
    if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(256) k_mb_read(const uint4 *__restrict__ p, long long n16, double *out)
{
    unsigned acc = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        uint4 q0, q1, q2, q3;
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(q0.x), "=r"(q0.y), "=r"(q0.z), "=r"(q0.w) : "l"(p + i));
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(q1.x), "=r"(q1.y), "=r"(q1.z), "=r"(q1.w) : "l"(p + i + stride));
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(q2.x), "=r"(q2.y), "=r"(q2.z), "=r"(q2.w) : "l"(p + i + 2 * stride));
        asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(q3.x), "=r"(q3.y), "=r"(q3.z), "=r"(q3.w) : "l"(p + i + 3 * stride));
        acc ^= q0.x ^ q0.y ^ q0.z ^ q0.w ^ q1.x ^ q1.y ^ q1.z ^ q1.w ^ q2.x ^ q2.y ^ q2.z ^ q2.w ^ q3.x ^ q3.y ^ q3.z ^ q3.w;
    }
    for (; i < n16; i += stride) { uint4 q = p[i]; acc ^= q.x ^ q.y ^ q.z ^ q.w; }
    if (acc == 0x12345u) out[0] = 1.0;
}

pwa_status run_microbench(pwa_ctx *ctx, int which, int64_t bytes, double *result)
{
    cudaEvent_t e0, e1;
    PWA_CUDA(ctx, cudaEventCreate(&e0));
    PWA_CUDA(ctx, cudaEventCreate(&e1));
    pwa_status s = ensure_scratch(ctx, which == 2 ? (size_t)bytes : 4096);
    if (s != PWA_OK) return s;
    double *out = ctx->d_result;
    const int iters = 4096;
    const int grid = ctx->sm_count * 8;
    float best = 1e30f;
    if (which == 2) PWA_CUDA(ctx, cudaMemsetAsync(ctx->d_scratch, 1, (size_t)bytes, ctx->stream));
    for (int rep = 0; rep < 7; ++rep) {
        PWA_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        if (which == 0) k_mb_dfma<<<grid, 256, 0, ctx->stream>>>(out, iters, 1.0);
        else if (which == 1) k_mb_dmma<<<grid, 256, 0, ctx->stream>>>(out, iters, 1.0);
        else if (which == 2) k_mb_read<<<ctx->sm_count * 8, 256, 0, ctx->stream>>>((const uint4 *)ctx->d_scratch, bytes / 16, out);
        else return fail(ctx, PWA_ERR_INVALID_ARG, "unknown microbench id");
        ctx->launches++;
        PWA_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
        PWA_CUDA(ctx, cudaEventSynchronize(e1));
        float ms = 0.f;
        PWA_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        if (rep >= 2 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    const double sec = best * 1e-3;
    if (which == 0) *result = 2.0 * 8.0 * iters * 256.0 * grid / sec * 1e-12;
    else if (which == 1) *result = 2.0 * 256.0 * 8.0 * iters * 8.0 * grid / sec * 1e-12;   // 8x8x4 MACs per warp mma
    else *result = (double)bytes / sec * 1e-9;
    return PWA_OK;
}

}  // namespace pwa
