// data_term_static.cu — pwa_data_term_static: the streaming data term (steps A2 - A5: S_i, ln I_i, A_ia / S_i, fp64
// reduction; eq. 1, eq. 3 first term) for callers that must not allocate: code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc.  It needs no pwa_ctx (creating one allocates).  The per-block
// partial slots and the ticket of the fixed-order reduction (reduce.cuh: block_finish) live in ONE file-scope
// `static __device__` array of a stated maximum size, which every GPU that loads libpwa.so holds until the process exits:
//
//     g_dt_static_scratch: 256 bytes (ticket) + kStaticMaxBlocks x (2 + 2 kStaticMaxWaves) doubles = 1 065 216 bytes
//
// In host code the array's name is only a stand-in for the symbol; the device address is fetched once per device with
// cudaGetSymbolAddress (with that device current) and handed to the kernel.  The entry point calls no cudaMalloc, cudaFree
// or allocating library routine: one cudaMemsetAsync of the 256-byte ticket area (it must start at zero) and one kernel
// launch on the caller's stream.  V travels as a kernel parameter.  All calls share the array, which keeps the last call's
// partials: calls that overlap on the GPU (two streams, two host threads) race and give wrong sums; calls on one stream
// are ordered and safe.
//
// The kernel is a variant of k_data_term_generic (data_term.cu): one event per thread, any n <= 64, V in shared memory,
// per-warp shuffle sums, per-block partial in a fixed slot, the last block (ticket) adds the slots in slot order and writes
// the data-term-only record {L_data, n_nonfinite, Re T_0, Im T_0, ...} (the record of pwa_data_term_enqueue).
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "pwa_internal.h"
#include "reduce.cuh"

namespace pwa {

constexpr int kStaticMaxWaves = 64;                 // == PWA_STATIC_MAX_WAVES (pwa.h)
constexpr int kStaticMaxBlocks = 1024;
constexpr int kStaticThreads = 128;
constexpr int kStaticNC = 2 + 2 * kStaticMaxWaves;  // components of a partial at the largest n
constexpr int kStaticHead = 32;                     // doubles in front of the partials: 256 bytes, the ticket lives there

static __device__ __align__(256) double g_dt_static_scratch[kStaticHead + kStaticMaxBlocks * kStaticNC];

template <typename ST>
__global__ void __launch_bounds__(kStaticThreads)
k_data_term_static(const ST *__restrict__ A, long long N, const __grid_constant__ VArg varg, FinishArgs fa)
{
    constexpr int THREADS = kStaticThreads, NWARPS = THREADS / 32;
    __shared__ double sV[2 * kStaticMaxWaves];
    __shared__ double s_acc[NWARPS * kStaticNC];      // per-warp sums; doubles as block_finish scratch (>= THREADS doubles)
    __shared__ double s_tot[kStaticNC];
    const int n = fa.n, NC = 2 + 2 * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int t = tid; t < 2 * n; t += THREADS) sV[t] = varg.v[t];
    for (int t = tid; t < NWARPS * NC; t += THREADS) s_acc[t] = 0.0;
    __syncthreads();
    double *acc = s_acc + warp * NC;
    const long long stride = (long long)gridDim.x * THREADS;
    const long long nround = (N + stride - 1) / stride;
    for (long long it = 0; it < nround; ++it) {
        const long long i = it * stride + (long long)blockIdx.x * THREADS + tid;
        const bool valid = i < N;
        const ST *row = A + (valid ? i : 0) * 2 * n;
        double sr = 0.0, si = 0.0;                                   // A2: S_i = sum_a V_a A_ia
        for (int a = 0; a < n; ++a) {
            const double ar = valid ? (double)row[2 * a] : 0.0, ai = valid ? (double)row[2 * a + 1] : 0.0;
            sr = fma(sV[2 * a], ar, sr); sr = fma(-sV[2 * a + 1], ai, sr);
            si = fma(sV[2 * a], ai, si); si = fma(sV[2 * a + 1], ar, si);
        }
        const double I = sr * sr + si * si;
        const double l = log(I), inv = 1.0 / I;                      // A3: ln I_i; A4: r_i = 1 / S_i = conj(S_i) / I_i
        double rr = sr * inv, rim = -si * inv, lv = l, bv = (!(I > 0.0) || !isfinite(l)) ? 1.0 : 0.0;
        if (!valid) { rr = 0.0; rim = 0.0; lv = 0.0; bv = 0.0; }
        lv = warp_sum(lv); bv = warp_sum(bv);
        if (lane == 0) { acc[0] += lv; acc[1] += bv; }
        for (int a = 0; a < n; ++a) {
            const double ar = valid ? (double)row[2 * a] : 0.0, ai = valid ? (double)row[2 * a + 1] : 0.0;
            double xr = ar * rr - ai * rim, xi = ar * rim + ai * rr;
            xr = warp_sum(xr); xi = warp_sum(xi);
            if (lane == 0) { acc[2 + 2 * a] += xr; acc[3 + 2 * a] += xi; }
        }
    }
    __syncthreads();
    for (int c = tid; c < NC; c += THREADS) {
        double t = 0.0;
        for (int w = 0; w < NWARPS; ++w) t += s_acc[w * NC + c];
        s_tot[c] = t;
    }
    __syncthreads();
    block_finish(s_tot, s_acc, sV, fa);                              // A5: fixed slots + ticket; fa.M == nullptr: data-term-only record
}

namespace {

struct StaticDev {
    bool ready = false;
    double *scratch = nullptr;      // DEVICE address of g_dt_static_scratch on this device
    int sm_count = 0;
};
StaticDev s_static_dev[64];
std::mutex s_static_mutex;

pwa_status static_fail(char *errbuf, int32_t len, pwa_status st, const char *msg)
{
    if (errbuf != nullptr && len > 0) snprintf(errbuf, (size_t)len, "%s", msg);
    return st;
}

pwa_status static_cuda_fail(char *errbuf, int32_t len, cudaError_t e, const char *what)
{
    cudaGetLastError();
    if (errbuf != nullptr && len > 0) snprintf(errbuf, (size_t)len, "%s: %s", what, cudaGetErrorString(e));
    return PWA_ERR_CUDA;
}

}  // namespace

}  // namespace pwa

using namespace pwa;

extern "C" pwa_status pwa_data_term_static(int32_t device, void *cuda_stream, pwa_dtype storage, int32_t n_waves,
                                           const void *amps_dev, int64_t n_events, const double *V,
                                           double *out_dev, char *errbuf, int32_t errbuf_len)
{
    if (errbuf != nullptr && errbuf_len > 0) errbuf[0] = 0;
    if (n_waves < 1) return static_fail(errbuf, errbuf_len, PWA_ERR_INVALID_ARG, "pwa_data_term_static: n_waves must be >= 1");
    if (n_waves > kStaticMaxWaves) {
        char msg[160];
        snprintf(msg, sizeof(msg), "pwa_data_term_static: n_waves = %d exceeds the static scratch (PWA_STATIC_MAX_WAVES = %d); use a pwa_ctx",
                 (int)n_waves, kStaticMaxWaves);
        return static_fail(errbuf, errbuf_len, PWA_ERR_UNSUPPORTED, msg);
    }
    if (storage != PWA_F64 && storage != PWA_F32) return static_fail(errbuf, errbuf_len, PWA_ERR_INVALID_ARG, "pwa_data_term_static: bad storage type");
    if (n_events < 0 || (n_events > 0 && amps_dev == nullptr) || V == nullptr || out_dev == nullptr)
        return static_fail(errbuf, errbuf_len, PWA_ERR_INVALID_ARG, "pwa_data_term_static: null argument or negative n_events");
    if (device < 0 || device >= 64) return static_fail(errbuf, errbuf_len, PWA_ERR_INVALID_ARG, "pwa_data_term_static: device must be in [0, 64)");
    for (int t = 0; t < 2 * n_waves; ++t)
        if (!isfinite(V[t])) return static_fail(errbuf, errbuf_len, PWA_ERR_INVALID_ARG, "pwa_data_term_static: V contains non-finite values");
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return static_cuda_fail(errbuf, errbuf_len, e, "pwa_data_term_static: cudaSetDevice");

    // set-up, once per device, with that device current: the DEVICE address of the static array
    StaticDev &sd = s_static_dev[device];
    {
        std::lock_guard<std::mutex> lock(s_static_mutex);
        if (!sd.ready) {
            double *p = nullptr;
            e = cudaGetSymbolAddress((void **)&p, g_dt_static_scratch);
            if (e != cudaSuccess || p == nullptr) return static_cuda_fail(errbuf, errbuf_len, e, "pwa_data_term_static: cudaGetSymbolAddress");
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
            if (e != cudaSuccess) return static_cuda_fail(errbuf, errbuf_len, e, "pwa_data_term_static: cudaDeviceGetAttribute");
            sd.scratch = p; sd.sm_count = sms > 0 ? sms : 1; sd.ready = true;
        }
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    long long grid = (n_events + kStaticThreads - 1) / kStaticThreads;
    const long long cap = (long long)sd.sm_count * 4 < kStaticMaxBlocks ? (long long)sd.sm_count * 4 : kStaticMaxBlocks;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;

    FinishArgs fa;
    fa.ticket = reinterpret_cast<unsigned *>(sd.scratch);           // first 256 bytes
    fa.partials = sd.scratch + kStaticHead;
    fa.n = n_waves; fa.M = nullptr; fa.out = out_dev;
    VArg varg;
    memset(&varg, 0, sizeof(varg));
    for (int t = 0; t < 2 * n_waves; ++t) varg.v[t] = V[t];

    // the ticket must start at zero whatever an earlier (possibly failed) call left there; the partial slots need no
    // clearing: every block writes its slot before the last block reads slots 0 .. grid - 1
    e = cudaMemsetAsync(sd.scratch, 0, kStaticHead * sizeof(double), stream);
    if (e != cudaSuccess) return static_cuda_fail(errbuf, errbuf_len, e, "pwa_data_term_static: cudaMemsetAsync");
    if (storage == PWA_F32)
        k_data_term_static<float><<<(unsigned)grid, kStaticThreads, 0, stream>>>(reinterpret_cast<const float *>(amps_dev), n_events, varg, fa);
    else
        k_data_term_static<double><<<(unsigned)grid, kStaticThreads, 0, stream>>>(reinterpret_cast<const double *>(amps_dev), n_events, varg, fa);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_cuda_fail(errbuf, errbuf_len, e, "pwa_data_term_static: kernel launch");
    return PWA_OK;
}
