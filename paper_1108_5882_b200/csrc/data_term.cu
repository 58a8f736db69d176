// data_term.cu — steps A2-A5 of the hot path: one pass over the N x n data amplitude
// matrix in HBM that produces L_data = sum_i ln|S_i|^2 and T_a = sum_i A_ia / S_i.
//   S_i = sum_a V_a A_ia,  I_i = |S_i|^2            eq. 1
//   l_i = ln I_i                                    eq. 3, first term
//   r_i = 1 / S_i,  t_ia = A_ia r_i                 gradient contribution
// The paper's own formulation stores an N x n^2 lookup table; this build streams
// the N x n matrix instead (n/2 times fewer bytes) and is HBM-bound.
//
// Thread mapping: G lanes share one event; lane j owns the 16-byte
// chunks j, j+G, ... of the row, so a warp load covers 32/G rows x (G*16) contiguous bytes
// (fully used 32-byte sectors, 128-bit loads).  Each group takes E events per step; the E
// partial coherent sums of a lane are combined with a transposing shuffle reduction so
// that lane e ends up owning S of event e, takes ONE log and ONE reciprocal for it, and
// broadcasts r_e back.  The row stays in registers between the two uses (one HBM read).
// fp32 storage: widened to fp64 on use (exact, C16); all arithmetic and sums are fp64.
#include "pwa_internal.h"
#include "reduce.cuh"
#include "stream_common.cuh"

namespace pwa {

// Transposing reduction over the E lowest lane bits followed by a butterfly over the
// remaining bits of the group: on return (sr[0], si[0]) of lane j is the complete S of
// event (j & (E-1)).
template <int G, int E>
__device__ __forceinline__ void group_transpose_reduce(double (&sr)[E], double (&si)[E], int j)
{
#pragma unroll
    for (int h = E / 2; h >= 1; h >>= 1) {
        const bool up = (j & h) != 0;
#pragma unroll
        for (int t = 0; t < h; ++t) {
            double keep_r = up ? sr[t + h] : sr[t], send_r = up ? sr[t] : sr[t + h];
            double keep_i = up ? si[t + h] : si[t], send_i = up ? si[t] : si[t + h];
            sr[t] = keep_r + shfl_xor_d(send_r, h);
            si[t] = keep_i + shfl_xor_d(send_i, h);
        }
    }
#pragma unroll
    for (int m = E; m < G; m <<= 1) {
        sr[0] += shfl_xor_d(sr[0], m);
        si[0] += shfl_xor_d(si[0], m);
    }
}

template <typename ST, int G, int CK, int E, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
k_data_term(const uint4 *__restrict__ A, long long N, VArg varg, FinishArgs fa, const double *__restrict__ wt)
{
    constexpr int WPC = Chunk<ST>::WPC;
    constexpr int W = CK * WPC;            // waves owned by a lane
    constexpr int CPR = G * CK;            // 16-byte chunks per row
    constexpr int NW = CPR * WPC;          // n
    constexpr int GPW = 32 / G;            // groups per warp
    constexpr int EPB = GPW * E;           // events per warp step
    constexpr int NWARPS = THREADS / 32;
    static_assert(E <= G && (G & (G - 1)) == 0 && (E & (E - 1)) == 0, "G, E powers of two, E <= G");

    __shared__ double sV[2 * NW];
    for (int t = threadIdx.x; t < 2 * NW; t += THREADS) sV[t] = varg.v[t];
    __syncthreads();

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = lane % G, grp = lane / G;

    double vr[W], vi[W], tr[W], ti[W];
#pragma unroll
    for (int k = 0; k < CK; ++k)
#pragma unroll
        for (int w = 0; w < WPC; ++w) {
            int a = (j + G * k) * WPC + w;
            vr[k * WPC + w] = sV[2 * a]; vi[k * WPC + w] = sV[2 * a + 1];
            tr[k * WPC + w] = 0.0; ti[k * WPC + w] = 0.0;
        }
    double L = 0.0, bad = 0.0;

    const long long nsteps = (N + EPB - 1) / EPB;
    for (long long b = (long long)blockIdx.x * NWARPS + warp; b < nsteps; b += (long long)gridDim.x * NWARPS) {
        const long long ev0 = b * EPB + (long long)grp * E;
        uint4 q[E][CK];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const long long row = ev0 + e;
#pragma unroll
            for (int k = 0; k < CK; ++k) {
                if (row < N) q[e][k] = ldg_stream(A + row * CPR + j + G * k);
                else         q[e][k] = make_uint4(0u, 0u, 0u, 0u);
            }
        }
        // A2: partial coherent sums over this lane's waves
        double sr[E], si[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            double ar[WPC], ai[WPC];
            sr[e] = 0.0; si[e] = 0.0;
#pragma unroll
            for (int k = 0; k < CK; ++k) {
                Chunk<ST>::unpack(q[e][k], ar, ai);
#pragma unroll
                for (int w = 0; w < WPC; ++w) {
                    sr[e] = fma(vr[k * WPC + w], ar[w], sr[e]); sr[e] = fma(-vi[k * WPC + w], ai[w], sr[e]);
                    si[e] = fma(vr[k * WPC + w], ai[w], si[e]); si[e] = fma(vi[k * WPC + w], ar[w], si[e]);
                }
            }
        }
        group_transpose_reduce<G, E>(sr, si, j);
        // A3 + A4 for the one event this lane owns
        const int my_e = j & (E - 1);
        const bool valid = (ev0 + my_e) < N;
        const double I = sr[0] * sr[0] + si[0] * si[0];
        const double l = log(I);
        const double inv = 1.0 / I;
        double rr = sr[0] * inv, rim = -si[0] * inv;      // r = conj(S) / I
        const bool counted = valid && (j < E);             // each event is owned by G/E lanes
        double wv = 1.0;                                   // NEXT-3: optional event weight, L = sum w l, T = sum w A / S
        if (wt != nullptr && valid) { wv = __ldg(wt + ev0 + my_e); rr *= wv; rim *= wv; }
        if (counted) { L += wv * l; if (!(I > 0.0) || !isfinite(l)) bad += 1.0; }
        if (!valid) { rr = 0.0; rim = 0.0; }
        // A4: t_ia = A_ia r_i accumulated into the lane's T
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double er = __shfl_sync(0xffffffffu, rr, e, G);
            const double ei = __shfl_sync(0xffffffffu, rim, e, G);
            double ar[WPC], ai[WPC];
#pragma unroll
            for (int k = 0; k < CK; ++k) {
                Chunk<ST>::unpack(q[e][k], ar, ai);
#pragma unroll
                for (int w = 0; w < WPC; ++w) {
                    tr[k * WPC + w] = fma(ar[w], er, tr[k * WPC + w]); tr[k * WPC + w] = fma(-ai[w], ei, tr[k * WPC + w]);
                    ti[k * WPC + w] = fma(ar[w], ei, ti[k * WPC + w]); ti[k * WPC + w] = fma(ai[w], er, ti[k * WPC + w]);
                }
            }
        }
    }
    auto wave_of = [&](int idx) { return (j + G * (idx / WPC)) * WPC + (idx % WPC); };
    reduce_and_finish<G, W, THREADS>(L, bad, tr, ti, wave_of, sV, fa);
}

// Generic fallback: any n <= kMaxWaves, thread per event, V from device memory.
template <typename ST, int THREADS>
__global__ void __launch_bounds__(THREADS)
k_data_term_generic(const ST *__restrict__ A, long long N, const double *__restrict__ Vdev, FinishArgs fa,
                    const double *__restrict__ wt)
{
    constexpr int NWARPS = THREADS / 32;
    extern __shared__ double dyn[];
    const int n = fa.n, NC = 2 + 2 * n;
    double *sV = dyn;                         // [2n]
    double *s_acc = dyn + 2 * n;              // [NWARPS][NC]
    double *s_tot = s_acc + (NWARPS * NC > THREADS ? NWARPS * NC : THREADS);   // [NC]; s_acc doubles as block_finish scratch (>= THREADS)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int t = tid; t < 2 * n; t += THREADS) sV[t] = Vdev[t];
    for (int t = tid; t < NWARPS * NC; t += THREADS) s_acc[t] = 0.0;
    __syncthreads();
    double *acc = s_acc + warp * NC;
    const long long stride = (long long)gridDim.x * THREADS;
    const long long nround = (N + stride - 1) / stride;
    for (long long it = 0; it < nround; ++it) {
        const long long i = it * stride + (long long)blockIdx.x * THREADS + tid;
        const bool valid = i < N;
        const ST *row = A + (valid ? i : 0) * 2 * n;
        double sr = 0.0, si = 0.0;
        for (int a = 0; a < n; ++a) {
            double ar = valid ? (double)row[2 * a] : 0.0, ai = valid ? (double)row[2 * a + 1] : 0.0;
            sr = fma(sV[2 * a], ar, sr); sr = fma(-sV[2 * a + 1], ai, sr);
            si = fma(sV[2 * a], ai, si); si = fma(sV[2 * a + 1], ar, si);
        }
        const double I = sr * sr + si * si;
        const double l = log(I), inv = 1.0 / I;
        double rr = sr * inv, rim = -si * inv, lv = l, bv = (!(I > 0.0) || !isfinite(l)) ? 1.0 : 0.0;
        if (!valid) { rr = 0.0; rim = 0.0; lv = 0.0; bv = 0.0; }
        else if (wt != nullptr) { const double wv = __ldg(wt + i); rr *= wv; rim *= wv; lv *= wv; }
        lv = warp_sum(lv); bv = warp_sum(bv);
        if (lane == 0) { acc[0] += lv; acc[1] += bv; }
        for (int a = 0; a < n; ++a) {
            double ar = valid ? (double)row[2 * a] : 0.0, ai = valid ? (double)row[2 * a + 1] : 0.0;
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
    block_finish(s_tot, s_acc, sV, fa);
}

template <typename ST, int G, int CK, int E, int THREADS, int MINB>
static pwa_status launch_fast(pwa_ctx *ctx, const VArg &varg, const FinishArgs &fa_in)
{
    auto kern = k_data_term<ST, G, CK, E, THREADS, MINB>;
    constexpr int EPB = (32 / G) * E, NWARPS = THREADS / 32;
    int occ = 0;
    PWA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const long long N = ctx->data.n_events;
    long long nsteps = (N + EPB - 1) / EPB;
    long long want = (nsteps + NWARPS - 1) / NWARPS;
    long long grid = (long long)ctx->sm_count * occ;
    if (want < grid) grid = want;
    if (grid < 1) grid = 1;
    FinishArgs fa = fa_in;
    pwa_status s = ensure_partials(ctx, (size_t)n_components(ctx->n) * (size_t)grid);
    if (s != PWA_OK) return s;
    fa.partials = ctx->d_partials;
    kern<<<(unsigned)grid, THREADS, 0, ctx->stream>>>((const uint4 *)ctx->data.amps, N, varg, fa, ctx->data.weights);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

template <typename ST>
static pwa_status launch_generic(pwa_ctx *ctx, const double *Vdev, const FinishArgs &fa_in)
{
    constexpr int THREADS = 128, NWARPS = THREADS / 32;
    const int n = ctx->n, NC = 2 + 2 * n;
    size_t smem = sizeof(double) * (size_t)(2 * n + (NWARPS * NC > THREADS ? NWARPS * NC : THREADS) + NC);
    auto kern = k_data_term_generic<ST, THREADS>;
    if (smem > 48 * 1024)
        PWA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const long long N = ctx->data.n_events;
    long long grid = (N + THREADS - 1) / THREADS;
    long long cap = (long long)ctx->sm_count * 4;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    FinishArgs fa = fa_in;
    pwa_status s = ensure_partials(ctx, (size_t)NC * (size_t)grid);
    if (s != PWA_OK) return s;
    fa.partials = ctx->d_partials;
    kern<<<(unsigned)grid, THREADS, smem, ctx->stream>>>((const ST *)ctx->data.amps, N, Vdev, fa, ctx->data.weights);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

pwa_status launch_factored_data_term(pwa_ctx *ctx, const double *Vk, const FinishArgs &fa);   // factored.cu
pwa_status launch_data_term_tma(pwa_ctx *ctx, const VArg &varg, const FinishArgs &fa, bool *handled, bool resident);   // data_term_tma.cu

// Starts the resident evaluation grid (data_term_tma.cu, RES): same kernel, same grid, same finish as a launched evaluation
// of record 0; *started stays false where the TMA kernel does not apply (the caller then evaluates by launches).
pwa_status launch_resident(pwa_ctx *ctx, bool *started)
{
    *started = false;
    const int n = ctx->n;
    if (ctx->data.factored || ctx->data.weights || ctx->opt_data_term != 0 || !(n == 4 || n == 8 || n == 16 || n == 32 || n == 64)) return PWA_OK;
    FinishArgs fa;
    fa.partials = nullptr; fa.ticket = ctx->d_ticket; fa.n = n;
    fa.M = ctx->d_M; fa.out = ctx->dev_result; fa.done_flag = ctx->dev_flags; fa.seq = ctx->seq;
    fa.tagged = ctx->dev_rres;
    fa.eq2 = ctx->opt_likelihood == 1; fa.n_eq2 = eq2_n_data(ctx);
    VArg varg;
    memset(&varg, 0, sizeof(varg));
    return launch_data_term_tma(ctx, varg, fa, started, true);
}

// V_host_k: host pointer to V of evaluation k (already staged in ctx->h_V, mirrored in d_V).
// out_dev_terms != nullptr selects the data-term-only output (multi-GPU path).
pwa_status launch_data_term(pwa_ctx *ctx, const double *V_host_k, int k, double *out_dev_terms)
{
    const int n = ctx->n;
    FinishArgs fa;
    fa.partials = nullptr;
    fa.ticket = ctx->d_ticket;
    fa.n = n;
    if (out_dev_terms) { fa.M = nullptr; fa.out = out_dev_terms; }
    else               { fa.M = ctx->d_M; fa.out = ctx->dev_result + (size_t)k * result_stride(n);
                         fa.done_flag = ctx->dev_flags + k; fa.seq = ctx->seq; }
    fa.eq2 = ctx->opt_likelihood == 1; fa.n_eq2 = eq2_n_data(ctx);

    if (ctx->data.factored) {
        if (ctx->data.weights) return fail(ctx, PWA_ERR_UNSUPPORTED, "event weights are not supported with factored (floating-resonance) uploads");
        return launch_factored_data_term(ctx, V_host_k, fa);
    }

    const bool f32 = ctx->storage == PWA_F32;
    const bool fast = (n == 4 || n == 8 || n == 16 || n == 32 || n == 64) && ctx->opt_data_term != 99;
    if (!fast) {
        const double *Vdev = ctx->d_V + (size_t)k * 2 * n;
        return f32 ? launch_generic<float>(ctx, Vdev, fa) : launch_generic<double>(ctx, Vdev, fa);
    }
    VArg varg;
    for (int t = 0; t < 2 * n; ++t) varg.v[t] = V_host_k[t];
    // "data_term": 0 = default: TMA-tiled two-phase kernel (data_term_tma.cu) where it applies (row of 128 .. 1024 bytes),
    // else the per-lane streaming kernel below; 20 = per-lane kernel always; 98 = default kernel
    // without programmatic dependent launch; 99 = generic kernel
    const bool per_lane = ctx->opt_data_term == 20;
    if (!per_lane) {
        bool handled = false;
        pwa_status s = launch_data_term_tma(ctx, varg, fa, &handled, false);
        if (s != PWA_OK || handled) return s;
    }
    //                           ST      G  CK  E  THREADS MINB
    if (!f32) {
        switch (n) {
        case 4:  return launch_fast<double, 2, 2, 2, 256, 2>(ctx, varg, fa);
        case 8:  return launch_fast<double, 4, 2, 4, 256, 2>(ctx, varg, fa);
        case 16: return launch_fast<double, 4, 4, 4, 256, 2>(ctx, varg, fa);
        case 32: return launch_fast<double, 8, 4, 4, 256, 2>(ctx, varg, fa);
        case 64: return launch_fast<double, 16, 4, 4, 256, 2>(ctx, varg, fa);
        }
    } else {
        switch (n) {
        case 4:  return launch_fast<float, 2, 1, 2, 256, 2>(ctx, varg, fa);
        case 8:  return launch_fast<float, 4, 1, 4, 256, 2>(ctx, varg, fa);
        case 16: return launch_fast<float, 4, 2, 4, 256, 2>(ctx, varg, fa);
        case 32: return launch_fast<float, 8, 2, 4, 256, 2>(ctx, varg, fa);
        case 64: return launch_fast<float, 16, 2, 4, 256, 2>(ctx, varg, fa);
        }
    }
    return fail(ctx, PWA_ERR_UNSUPPORTED, "data term: unsupported n");
}

}  // namespace pwa
