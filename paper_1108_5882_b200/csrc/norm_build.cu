// norm_build.cu — step A6: the normalisation matrix of eq. 3's second term (P:41 inner
// bracket; pre-calculated once when masses and widths are fixed, rebuilt every
// iteration when they float):
//     M_ab = (1/N_gen) sum_j conj(B_ja) B_jb        (index convention C1: Norm = V^H M V)
// Hermitian, so only blocks with a-block <= b-block are accumulated and the lower triangle
// is written as the conjugate.  Accumulation is fp64; fp32-stored amplitudes are widened
// exactly (C16).  In factored mode the tile producer recomputes
// B_ja = BW(m_j; M_r(a), G_r(a)) * Z_{j,s(a)} (step A1, C3) and nothing is written to HBM.
//
// This file holds the generic CUDA-core path (any n <= kMaxWaves): each CTA owns a strided
// set of event tiles, stages ET events in shared memory as fp64, and every thread keeps a
// 4 x 4 complex block of M in registers.  Per-CTA partials go to a fixed slot; a second
// kernel sums the slots in slot order (bitwise reproducible) and scales by 1/N_gen.
// The tensor-core (FP64 DMMA) path lives in norm_dmma.cu.
#include "pwa_internal.h"
#include "factored.cuh"

namespace pwa {

constexpr int NB_THREADS = 256;
constexpr int NB_ET = 32;            // events per smem tile

template <typename ST, bool FACT>
__global__ void __launch_bounds__(NB_THREADS)
k_norm_generic(const ST *__restrict__ B, long long N, int n, int nb, int total_pairs,
               FactArgs fargs, double *__restrict__ scratch)
{
    extern __shared__ double2 smem2[];
    const int tid = threadIdx.x;
    const int np = nb * 4;
    double2 *tile = smem2;                                   // [NB_ET][np]
    // pairs handled by this CTA: [pair0, pair0 + npairs)
    const int pair0 = blockIdx.y * NB_THREADS;
    const int npairs = min(NB_THREADS, total_pairs - pair0);
    const int nslices = NB_THREADS / npairs;
    const int p = tid % npairs, slice = tid / npairs;
    const bool active = slice < nslices;
    // pair index -> (ba <= bb), row-major over the upper triangle
    int ba = 0, bb = 0;
    {
        int q = pair0 + p, row = 0;
        while (q >= nb - row) { q -= nb - row; ++row; }
        ba = row; bb = row + q;
    }
    double accr[4][4], acci[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) { accr[i][j] = 0.0; acci[i][j] = 0.0; }

    const long long ntiles = (N + NB_ET - 1) / NB_ET;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const long long base = t * NB_ET;
        for (int idx = tid; idx < NB_ET * np; idx += NB_THREADS) {
            const int e = idx / np, a = idx % np;
            const long long ev = base + e;
            double2 v = make_double2(0.0, 0.0);
            if (ev < N && a < n) {
                if (FACT) {
                    v = factored_amp<ST>(fargs, ev, a);
                } else {
                    v.x = (double)B[(ev * n + a) * 2];
                    v.y = (double)B[(ev * n + a) * 2 + 1];
                }
            }
            tile[e * np + a] = v;
        }
        __syncthreads();
        if (active) {
            for (int e = slice; e < NB_ET; e += nslices) {
                double2 xa[4], xb[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) { xa[i] = tile[e * np + ba * 4 + i]; xb[i] = tile[e * np + bb * 4 + i]; }
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) {   // conj(a) * b
                        accr[i][j] = fma(xa[i].x, xb[j].x, accr[i][j]); accr[i][j] = fma(xa[i].y, xb[j].y, accr[i][j]);
                        acci[i][j] = fma(xa[i].x, xb[j].y, acci[i][j]); acci[i][j] = fma(-xa[i].y, xb[j].x, acci[i][j]);
                    }
            }
        }
        __syncthreads();
    }
    // cross-slice reduction in fixed slice order, 8 accumulators per round
    double *red = reinterpret_cast<double *>(smem2);          // [NB_THREADS][8]
    double *dst = scratch + ((size_t)blockIdx.x * total_pairs + pair0 + p) * 32;
#pragma unroll
    for (int round = 0; round < 4; ++round) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int i = round, j = c >> 1;
            red[tid * 8 + c] = (c & 1) ? acci[i][j] : accr[i][j];
        }
        __syncthreads();
        if (slice == 0) {
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                double s = 0.0;
                for (int sl = 0; sl < nslices; ++sl) s += red[(sl * npairs + p) * 8 + c];
                dst[round * 8 + c] = s;
            }
        }
        __syncthreads();
    }
}

// Sums the per-CTA slots in slot order, scales by 1/N_gen, writes both triangles.
__global__ void k_norm_finalize(const double *__restrict__ scratch, int nslots, int n, int nb,
                                int total_pairs, double inv_ngen, double *__restrict__ M)
{
    const int gid = blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total_pairs * 16) return;
    const int pair = gid / 16, ij = gid % 16, i = ij / 4, j = ij % 4;
    int q = pair, row = 0;
    while (q >= nb - row) { q -= nb - row; ++row; }
    const int ba = row, bb = row + q;
    const int a = ba * 4 + i, b = bb * 4 + j;
    if (a >= n || b >= n) return;
    if (ba == bb && i > j) return;                       // mirrored from (j, i)
    double re = 0.0, im = 0.0;
    for (int s = 0; s < nslots; ++s) {
        const double *src = scratch + ((size_t)s * total_pairs + pair) * 32 + ij * 2;
        re += src[0]; im += src[1];
    }
    re *= inv_ngen; im *= inv_ngen;
    if (a == b) im = 0.0;                                // |B_ja|^2 is real
    M[((size_t)a * n + b) * 2] = re;  M[((size_t)a * n + b) * 2 + 1] = im;
    if (a != b) { M[((size_t)b * n + a) * 2] = re;  M[((size_t)b * n + a) * 2 + 1] = -im; }
}

pwa_status launch_norm_dmma(pwa_ctx *ctx, bool *handled);   // norm_dmma.cu

static pwa_status launch_norm_generic(pwa_ctx *ctx)
{
    const int n = ctx->n, nb = (n + 3) / 4, total_pairs = nb * (nb + 1) / 2;
    const long long N = ctx->mc.n_events;
    const long long ntiles = (N + NB_ET - 1) / NB_ET;
    long long gx = (long long)ctx->sm_count * 2;
    if (gx > ntiles) gx = ntiles;
    if (gx < 1) gx = 1;
    const int gy = (total_pairs + NB_THREADS - 1) / NB_THREADS;
    size_t smem = sizeof(double2) * (size_t)NB_ET * (size_t)nb * 4;
    if (smem < sizeof(double) * NB_THREADS * 8) smem = sizeof(double) * NB_THREADS * 8;
    pwa_status s = ensure_scratch(ctx, sizeof(double) * (size_t)gx * (size_t)total_pairs * 32);
    if (s != PWA_OK) return s;
    FactArgs fargs;
    const bool fact = ctx->mc.factored;
    if (fact) {
        s = fill_fact_args(ctx, ctx->mc, &fargs);
        if (s != PWA_OK) return s;
    } else {
        memset(&fargs, 0, sizeof(fargs));
    }
    dim3 grid((unsigned)gx, (unsigned)gy);
    const bool f32 = ctx->storage == PWA_F32;
#define LAUNCH_NB(ST, FACT)                                                                        \
    do {                                                                                           \
        auto kern = k_norm_generic<ST, FACT>;                                                      \
        if (smem > 48 * 1024)                                                                      \
            PWA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,  \
                                               (int)smem));                                        \
        kern<<<grid, NB_THREADS, smem, ctx->stream>>>((const ST *)ctx->mc.amps, N, n, nb,          \
                                                      total_pairs, fargs, ctx->d_scratch);         \
    } while (0)
    if (fact) { if (f32) LAUNCH_NB(float, true); else LAUNCH_NB(double, true); }
    else      { if (f32) LAUNCH_NB(float, false); else LAUNCH_NB(double, false); }
#undef LAUNCH_NB
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    const int fthreads = 128, fblocks = (total_pairs * 16 + fthreads - 1) / fthreads;
    k_norm_finalize<<<fblocks, fthreads, 0, ctx->stream>>>(ctx->d_scratch, (int)gx, n, nb, total_pairs,
                                                           1.0 / (double)ctx->mc.n_gen, ctx->d_M);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

pwa_status launch_norm_build(pwa_ctx *ctx)
{
    ctx->M_path = 0;
    if (ctx->mc.n_events == 0) {   // empty MC sample: M = 0
        PWA_CUDA(ctx, cudaMemsetAsync(ctx->d_M, 0, sizeof(double) * 2 * (size_t)ctx->n * ctx->n, ctx->stream));
        return PWA_OK;
    }
    // opt_norm: 0 = default (int8 tensor-core path for large fp32-stored samples, else FP64 DMMA),
    //           1 = FP64 DMMA, 2 = int8 tcgen05 path whenever the shape allows, 99 = generic CUDA-core kernel
    //           3 = int8 tcgen05 path with THREE digit planes (24 bits below the column maximum: faster, larger a-priori bound)
    if (ctx->opt_norm == 2 || ctx->opt_norm == 3 || (ctx->opt_norm == 0 && ctx->mc.n_events >= 65536)) {
        bool handled = false;
        pwa_status s = launch_norm_i8(ctx, &handled, ctx->opt_norm == 3);
        if (s != PWA_OK) return s;
        if (handled) { ctx->M_path = ctx->opt_norm == 3 ? 3 : 1; return PWA_OK; }
    }
    if (ctx->opt_norm != 99) {
        bool handled = false;
        pwa_status s = launch_norm_dmma(ctx, &handled);
        if (s != PWA_OK) return s;
        if (handled) return PWA_OK;
    }
    if (ctx->mc.weights) return fail(ctx, PWA_ERR_UNSUPPORTED, "MC event weights need n <= 64 (FP64 DMMA path)");
    return launch_norm_generic(ctx);
}

}  // namespace pwa
