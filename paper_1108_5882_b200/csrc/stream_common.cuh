// stream_common.cuh — device helpers shared by the streaming data-pass kernels: 128-bit
// streaming loads, the 16-byte chunk -> (re, im) unpacking for fp64 / fp32 storage (C16: fp32 is
// widened exactly, everything after the load is fp64), and the mbarrier / bulk-copy (TMA) PTX.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pwa {

__device__ __forceinline__ uint4 ldg_stream(const uint4 *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

template <typename ST> struct Chunk;
template <> struct Chunk<double> {
    static constexpr int WPC = 1;   // waves per 16-byte chunk
    static __device__ __forceinline__ void unpack(const uint4 &q, double *re, double *im)
    {
        re[0] = __hiloint2double((int)q.y, (int)q.x);
        im[0] = __hiloint2double((int)q.w, (int)q.z);
    }
};
template <> struct Chunk<float> {
    static constexpr int WPC = 2;
    static __device__ __forceinline__ void unpack(const uint4 &q, double *re, double *im)
    {
        re[0] = (double)__uint_as_float(q.x); im[0] = (double)__uint_as_float(q.y);
        re[1] = (double)__uint_as_float(q.z); im[1] = (double)__uint_as_float(q.w);
    }
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
                 "selp.u32 %0, 1, 0, p;\n"
                 "}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// try_wait suspends the thread for a hardware time slice per call; a copy that never completes
// (a corrupt descriptor) traps after ~2^26 slices instead of hanging the device.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    if (mbar_try_wait(bar, parity)) return;
    unsigned spins = 0;
    while (!mbar_try_wait(bar, parity)) { if (++spins > (1u << 26)) __trap(); }
}
__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}


}  // namespace pwa
