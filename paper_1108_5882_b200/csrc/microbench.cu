// microbench.cu — register-resident peak probes used as roofline denominators
// (MEASURED_PEAKS.json has no fp64 figure): fp64 FMA, fp64 mma.sync m8n8k4, HBM read stream.
#include "pwa_internal.h"
#include "tcgen05_common.cuh"

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

// int8 tensor-core probe: one CTA per SM issues `iters` x 4 tcgen05.mma.kind::i8 (M = 128, N, K = 32, both operands
// K-major digit planes in shared memory, whatever bytes they hold) into one TMEM accumulator and waits for the commit.
template <int N>
__global__ void __launch_bounds__(128, 1) k_mb_umma(int iters, double *out)
{
    extern __shared__ unsigned char mb_smem[];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t tmem_base_s;
    const uint32_t base = (smem_u32(mb_smem) + 1023u) & ~1023u;
    if (threadIdx.x == 0) { mbar_init(smem_u32(&bar), 1); tc::fence_async_smem(); }
    if (threadIdx.x < 32) tc::tmem_alloc(smem_u32(&tmem_base_s), 512);
    tc::tc_fence_before();
    __syncthreads();
    tc::tc_fence_after();
    const uint32_t tmem0 = tmem_base_s;
    if (threadIdx.x == 0) {
        constexpr uint32_t id = tc::idesc_i8(N, false, false);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
                tc::umma_i8(tmem0 + (uint32_t)((it & 1) * 256), tc::desc_kmajor(base + 32u * kk), tc::desc_kmajor(base + 16384u + 32u * kk), id, 1u);
        }
        tc::umma_commit(smem_u32(&bar));
        mbar_wait(smem_u32(&bar), 0);
    }
    tc::tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) { tc::tc_fence_after(); tc::tmem_dealloc(tmem0, 512); }
    if (out == nullptr) return;
}

// TMEM read probe: 16 warps (4 per lane quarter) loop over tcgen05.ld 32x32b.x16 of their quarter
__global__ void __launch_bounds__(512, 1) k_mb_tmem_ld(int iters, double *out)
{
    __shared__ uint32_t tmem_base_s;
    if (threadIdx.x < 32) tc::tmem_alloc(smem_u32(&tmem_base_s), 512);
    tc::tc_fence_before();
    __syncthreads();
    tc::tc_fence_after();
    const uint32_t tmem0 = tmem_base_s;
    const int warp = threadIdx.x >> 5, q = warp & 3, j = warp >> 2;
    int acc = 0;
    for (int it = 0; it < iters; ++it) {
        int32_t v[16];
        tc::tmem_ld16(tmem0 + ((uint32_t)(32 * q) << 16) + (uint32_t)(128 * j + 16 * (it & 7)), v);
        tc::tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 16; ++i) acc ^= v[i];
    }
    if (acc == 0x12345 && out != nullptr) out[0] = 1.0;
    tc::tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) { tc::tc_fence_after(); tc::tmem_dealloc(tmem0, 512); }
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
        else if (which == 3 || which == 4 || which == 5 || which == 6) {
            constexpr int SM = 1024 + 16384 + 32768;
            if (rep == 0) {
                PWA_CUDA(ctx, cudaFuncSetAttribute(k_mb_umma<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM));
                PWA_CUDA(ctx, cudaFuncSetAttribute(k_mb_umma<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM));
                PWA_CUDA(ctx, cudaFuncSetAttribute(k_mb_umma<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM));
                PWA_CUDA(ctx, cudaFuncSetAttribute(k_mb_umma<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SM));
            }
            if (which == 3) k_mb_umma<256><<<ctx->sm_count, 128, SM, ctx->stream>>>(iters, nullptr);
            else if (which == 4) k_mb_umma<128><<<ctx->sm_count, 128, SM, ctx->stream>>>(iters, nullptr);
            else if (which == 5) k_mb_umma<64><<<ctx->sm_count, 128, SM, ctx->stream>>>(iters, nullptr);
            else k_mb_umma<32><<<ctx->sm_count, 128, SM, ctx->stream>>>(iters, nullptr);
        }
        else if (which == 7) k_mb_tmem_ld<<<ctx->sm_count, 512, 0, ctx->stream>>>(iters * 4, nullptr);
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
    else if (which >= 3 && which <= 6) {                                                    // int8 Top/s
        const double N = which == 3 ? 256.0 : which == 4 ? 128.0 : which == 5 ? 64.0 : 32.0;
        *result = 2.0 * 128.0 * N * 32.0 * 4.0 * iters * ctx->sm_count / sec * 1e-12;
    }
    else if (which == 7) *result = 16.0 * 32.0 * 16.0 * 4.0 * (iters * 4.0) * ctx->sm_count / sec * 1e-9;   // GB/s of TMEM reads
    else *result = (double)bytes / sec * 1e-9;
    return PWA_OK;
}

}  // namespace pwa
