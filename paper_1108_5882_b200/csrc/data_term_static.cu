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
// The kernel is a variant of the per-lane streaming kernel (data_term.cu) for any n <= 64: a group of lanes shares an event,
// every lane keeps the T sums of its own waves, per-block partial in a fixed slot, the last block (ticket) adds the slots
// in slot order and writes the data-term-only record {L_data, n_nonfinite, Re T_0, Im T_0, ...} (the record of
// pwa_data_term_enqueue).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
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

// G = (next power of two >= n) / 4 adjacent lanes share an event, lane j of a group owns the W = 4 waves j, j + G, ..:
// 8- / 16-byte loads of one complex amplitude per lane and wave, partial S_i combined with an xor-shuffle tree over the
// group, then every lane adds A_ia / S_i of its own waves to its private T accumulators (no cross-lane sum per event).
// E events per group are in flight per step.  At the end the 32 / G groups of a warp are summed with xor shuffles, the
// warps in shared memory, the blocks through fixed slots + ticket (block_finish): bitwise reproducible for a fixed shape.
template <typename ST> struct StaticLoad;
template <> struct StaticLoad<float> {
    static __device__ __forceinline__ double2 ld(const float *row, int a) { const float2 v = __ldg(reinterpret_cast<const float2 *>(row) + a); return make_double2((double)v.x, (double)v.y); }
};
template <> struct StaticLoad<double> {
    static __device__ __forceinline__ double2 ld(const double *row, int a) { return __ldg(reinterpret_cast<const double2 *>(row) + a); }
};

template <typename ST, int G, int W>
__global__ void __launch_bounds__(kStaticThreads)
k_data_term_static(const ST *__restrict__ A, long long N, const __grid_constant__ VArg varg, FinishArgs fa)
{
    constexpr int THREADS = kStaticThreads, NWARPS = THREADS / 32, GPW = 32 / G, E = 4, EPS = GPW * E;   // events per warp step
    __shared__ double sV[2 * kStaticMaxWaves];
    __shared__ double s_acc[NWARPS * kStaticNC];      // per-warp sums; doubles as block_finish scratch (>= THREADS doubles)
    __shared__ double s_tot[kStaticNC];
    const int n = fa.n, NC = 2 + 2 * n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int j = lane % G, grp = lane / G;
    for (int t = tid; t < 2 * n; t += THREADS) sV[t] = varg.v[t];
    __syncthreads();
    double vr[W], vi[W], tr[W], ti[W];
#pragma unroll
    for (int w = 0; w < W; ++w) {
        const int a = j + G * w;
        vr[w] = a < n ? sV[2 * a] : 0.0; vi[w] = a < n ? sV[2 * a + 1] : 0.0;
        tr[w] = 0.0; ti[w] = 0.0;
    }
    double L = 0.0, bad = 0.0;
    const long long nsteps = (N + EPS - 1) / EPS;
    for (long long st = (long long)blockIdx.x * NWARPS + warp; st < nsteps; st += (long long)gridDim.x * NWARPS) {
        double2 x[E][W];
        double sr[E], si[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const long long i = st * EPS + (long long)grp * E + e;
#pragma unroll
            for (int w = 0; w < W; ++w) {
                const int a = j + G * w;
                x[e][w] = (i < N && a < n) ? StaticLoad<ST>::ld(A + i * 2 * n, a) : make_double2(0.0, 0.0);
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            sr[e] = 0.0; si[e] = 0.0;
#pragma unroll
            for (int w = 0; w < W; ++w) {                            // A2: S_i = sum_a V_a A_ia
                sr[e] = fma(vr[w], x[e][w].x, sr[e]); sr[e] = fma(-vi[w], x[e][w].y, sr[e]);
                si[e] = fma(vr[w], x[e][w].y, si[e]); si[e] = fma(vi[w], x[e][w].x, si[e]);
            }
#pragma unroll
            for (int m = 1; m < G; m <<= 1) { sr[e] += shfl_xor_d(sr[e], m); si[e] += shfl_xor_d(si[e], m); }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const long long i = st * EPS + (long long)grp * E + e;
            if (i < N) {                                             // uniform over the group
                const double I = sr[e] * sr[e] + si[e] * si[e];
                const double inv = 1.0 / I;                          // A4: r_i = 1 / S_i = conj(S_i) / I_i
                const double rr = sr[e] * inv, rim = -si[e] * inv;
                if (j == 0) {
                    const double l = log(I);                         // A3: ln I_i
                    L += l;
                    if (!(I > 0.0) || !isfinite(l)) bad += 1.0;
                }
#pragma unroll
                for (int w = 0; w < W; ++w) {
                    tr[w] += x[e][w].x * rr - x[e][w].y * rim;
                    ti[w] += x[e][w].x * rim + x[e][w].y * rr;
                }
            }
        }
    }
    // groups of the warp -> lanes 0 .. G - 1
#pragma unroll
    for (int m = G; m < 32; m <<= 1) {
        L += shfl_xor_d(L, m); bad += shfl_xor_d(bad, m);
#pragma unroll
        for (int w = 0; w < W; ++w) { tr[w] += shfl_xor_d(tr[w], m); ti[w] += shfl_xor_d(ti[w], m); }
    }
    double *acc = s_acc + warp * NC;
    if (lane == 0) { acc[0] = L; acc[1] = bad; }
    if (lane < G) {
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int a = j + G * w;
            if (a < n) { acc[2 + 2 * a] = tr[w]; acc[3 + 2 * a] = ti[w]; }
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

template <typename ST, int G, int W>
static cudaError_t launch_static(const void *amps, long long N, const VArg &varg, const FinishArgs &fa, int sm_count, cudaStream_t stream)
{
    constexpr int EPS = (32 / G) * 4, NWARPS = kStaticThreads / 32;
    long long grid = ((N + EPS - 1) / EPS + NWARPS - 1) / NWARPS;
    const long long cap = (long long)sm_count * 6 < kStaticMaxBlocks ? (long long)sm_count * 6 : kStaticMaxBlocks;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    k_data_term_static<ST, G, W><<<(unsigned)grid, kStaticThreads, 0, stream>>>(reinterpret_cast<const ST *>(amps), N, varg, fa);
    return cudaGetLastError();
}

template <typename ST>
static cudaError_t dispatch_static(int n, const void *amps, long long N, const VArg &varg, const FinishArgs &fa, int sm_count, cudaStream_t stream)
{
    // up to W = 4 waves per lane: G = (next power of two >= n) / 4 lanes per event
    if (n > 32) return launch_static<ST, 16, 4>(amps, N, varg, fa, sm_count, stream);
    if (n > 16) return launch_static<ST, 8, 4>(amps, N, varg, fa, sm_count, stream);
    if (n > 8)  return launch_static<ST, 4, 4>(amps, N, varg, fa, sm_count, stream);
    if (n > 4)  return launch_static<ST, 2, 4>(amps, N, varg, fa, sm_count, stream);
    return launch_static<ST, 1, 4>(amps, N, varg, fa, sm_count, stream);
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
    if ((reinterpret_cast<uintptr_t>(amps_dev) & 15u) != 0 || (reinterpret_cast<uintptr_t>(out_dev) & 7u) != 0)
        return static_fail(errbuf, errbuf_len, PWA_ERR_INVALID_ARG, "pwa_data_term_static: amps_dev must be 16-byte aligned, out_dev 8-byte aligned");
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
    e = storage == PWA_F32 ? dispatch_static<float>(n_waves, amps_dev, n_events, varg, fa, sd.sm_count, stream)
                           : dispatch_static<double>(n_waves, amps_dev, n_events, varg, fa, sd.sm_count, stream);
    if (e != cudaSuccess) return static_cuda_fail(errbuf, errbuf_len, e, "pwa_data_term_static: kernel launch");
    return PWA_OK;
}
