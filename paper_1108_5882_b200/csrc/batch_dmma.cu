// batch_dmma.cu — step A8 on the FP64 tensor cores: K starting points
// V_k evaluated in ONE pass over the data amplitudes ("fits are usually repeated with
// various sets of starting parameters").  Per tile of E events, with X = the interleaved
// (re, im) amplitude rows viewed as a real [E x D] matrix (D = 2n):
//   GEMM1   S = X W          W[2a][2k] = Re V, W[2a+1][2k] = -Im V, W[2a][2k+1] = Im V, W[2a+1][2k+1] = Re V
//                            -> S[e][2k] = Re S_ek, S[e][2k+1] = Im S_ek           (eq. 1)
//   epilogue l_k += ln|S_ek|^2 ;  R_ek = 1 / S_ek = conj(S_ek)/|S_ek|^2            (eq. 3 first term)
//   GEMM2   Q = X^T Rm       Rm[e][2k] = Re R, Rm[e][2k+1] = Im R
//                            -> Re T_ak = Q[2a][2k] - Q[2a+1][2k+1],  Im T_ak = Q[2a][2k+1] + Q[2a+1][2k]
// S and R never touch HBM.  tcgen05.mma has no f64 kind, so both GEMMs are warp-level
// mma.sync.m8n8k4.f64 (DMMA); operands come from padded shared-memory tiles (row strides = 4 mod
// 16 doubles: conflict-free fragment loads), the GEMM2 accumulators (the whole D x 2KC block of
// Q) stay in registers for the CTA's event range.  KC = 32 starting points per pass (W = D x 64
// doubles in smem); K > 32 takes ceil(K/32) passes over A (the path is DMMA-bound by ~10x, so the
// extra HBM reads are hidden).  Per-CTA partials go to fixed slots; k_batch_finalize sums them in
// slot order and performs step A7 per column.
#include "pwa_internal.h"
#include "reduce.cuh"

namespace pwa {

constexpr int BD_THREADS = 256;       // 8 warps
constexpr int BD_E = 64;              // events per tile
constexpr int BD_KC = 32;             // starting points per pass
constexpr int BD_C = 2 * BD_KC;       // real columns per pass (8 column blocks)
constexpr int BD_CP = BD_C + 4;       // padded row stride of W and R tiles (doubles)

__device__ __forceinline__ void bd_dmma(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ uint4 bd_ldg16(const uint4 *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

template <int NB> struct BatchCfg {
    static constexpr int D = NB * 8, XP = D + 4;
    // GEMM2 warp grid: WR row-block groups x WC column-block groups (8 warps)
    static constexpr int WR = NB >= 4 ? 4 : (NB == 2 ? 2 : 1), WC = 8 / WR;
    static constexpr int RB = NB / WR, CB = 8 / WC;
    static constexpr size_t SMEM = sizeof(double) * ((size_t)D * BD_CP + (size_t)BD_E * XP + (size_t)BD_E * BD_CP + 2 * BD_KC * 4);
};

// scratch per slot (= CTA): Q blocks [NB][8][64] doubles, then L[KC], bad[KC]
__host__ __device__ inline size_t bd_slot_doubles(int NB) { return (size_t)NB * 8 * 64 + 2 * BD_KC; }

template <typename ST, int NB, bool ALIGNED>
__global__ void __launch_bounds__(BD_THREADS, 1)
k_batch_dmma(const void *__restrict__ Av, long long N, int n, const double *__restrict__ Vdev, int K, int k0,
             double *__restrict__ scratch)
{
    using C = BatchCfg<NB>;
    constexpr int D = C::D, XP = C::XP, WR = C::WR, WC = C::WC, RB = C::RB, CB = C::CB;
    constexpr int CH = 16 / (int)sizeof(ST), RC = D / CH, CPT = (BD_E * RC + BD_THREADS - 1) / BD_THREADS;
    extern __shared__ double bd_smem[];
    double *sW = bd_smem;                         // [D][BD_CP]
    double *sX = sW + D * BD_CP;                  // [BD_E][XP]
    double *sR = sX + BD_E * XP;                  // [BD_E][BD_CP]
    double *sL = sR + BD_E * BD_CP;               // [4][2 * BD_KC]  (L and bad, per GEMM1 event-row group)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lq = lane >> 2, lr = lane & 3;

    // ---- W from V (columns k0 .. k0+KC-1; columns past K replicate column k0 and are discarded)
    for (int idx = tid; idx < D * BD_C; idx += BD_THREADS) {
        const int d = idx / BD_C, c = idx % BD_C;
        const int a = d >> 1, p = d & 1, kl = c >> 1, q = c & 1;
        int k = k0 + kl; if (k >= K) k = k0;
        double w = 0.0;
        if (a < n) {
            const double vr = Vdev[((size_t)k * n + a) * 2], vi = Vdev[((size_t)k * n + a) * 2 + 1];
            w = (p == q) ? vr : (p == 1 ? -vi : vi);
        }
        sW[d * BD_CP + c] = w;
    }

    // GEMM1 partition: 4 event-row groups (2 event blocks each) x 2 column groups (4 column blocks each)
    const int er = warp >> 1, cg = warp & 1;
    // GEMM2 partition
    const int rg = warp / WC, cg2 = warp % WC;

    double q2[RB][CB][2];
#pragma unroll
    for (int i = 0; i < RB; ++i)
#pragma unroll
        for (int j = 0; j < CB; ++j) { q2[i][j][0] = 0.0; q2[i][j][1] = 0.0; }
    double Lacc[4] = {0.0, 0.0, 0.0, 0.0}, badacc[4] = {0.0, 0.0, 0.0, 0.0};

    const long long ntiles = (N + BD_E - 1) / BD_E;
    uint4 stage[CPT];
    auto load_tile = [&](long long t) {
        if constexpr (ALIGNED) {
#pragma unroll
            for (int c = 0; c < CPT; ++c) {
                const int idx = tid + c * BD_THREADS;
                const int e = idx / RC, ch = idx % RC;
                const long long ev = t * BD_E + e;
                if (idx < BD_E * RC && ev < N) stage[c] = bd_ldg16(reinterpret_cast<const uint4 *>(Av) + ev * RC + ch);
                else                           stage[c] = make_uint4(0u, 0u, 0u, 0u);
            }
        }
    };
    auto store_tile = [&](long long t) {
        if constexpr (ALIGNED) {
#pragma unroll
            for (int c = 0; c < CPT; ++c) {
                const int idx = tid + c * BD_THREADS;
                if (idx >= BD_E * RC) continue;
                const int e = idx / RC, ch = idx % RC;
                double *d = sX + e * XP + ch * CH;
                if (sizeof(ST) == 8) {
                    *reinterpret_cast<double2 *>(d) = make_double2(__hiloint2double((int)stage[c].y, (int)stage[c].x),
                                                                   __hiloint2double((int)stage[c].w, (int)stage[c].z));
                } else {
                    *reinterpret_cast<double2 *>(d) = make_double2((double)__uint_as_float(stage[c].x), (double)__uint_as_float(stage[c].y));
                    *reinterpret_cast<double2 *>(d + 2) = make_double2((double)__uint_as_float(stage[c].z), (double)__uint_as_float(stage[c].w));
                }
            }
        } else {
            const ST *A = reinterpret_cast<const ST *>(Av);
            const int d2 = 2 * n;
            for (int idx = tid; idx < BD_E * D; idx += BD_THREADS) {
                const int e = idx / D, c = idx % D;
                const long long ev = t * BD_E + e;
                sX[e * XP + c] = (ev < N && c < d2) ? (double)A[ev * d2 + c] : 0.0;
            }
        }
    };

    long long t = blockIdx.x;
    if (t < ntiles) load_tile(t);
    for (; t < ntiles; t += gridDim.x) {
        __syncthreads();                       // previous tile fully consumed (sX, sR free); W ready
        store_tile(t);
        const long long nxt = t + gridDim.x;
        if (nxt < ntiles) load_tile(nxt);      // prefetch into registers, lands during the GEMMs
        __syncthreads();

        // ---------------- GEMM1: S[2 event blocks][4 column blocks] over D
        double s1[2][4][2];
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
            for (int c = 0; c < 4; ++c) { s1[m][c][0] = 0.0; s1[m][c][1] = 0.0; }
        {
            const double *xa = sX + ((er * 2) * 8 + lq) * XP + lr;
            const double *wb = sW + lr * BD_CP + (cg * 4) * 8 + lq;
#pragma unroll 4
            for (int ks = 0; ks < D / 4; ++ks) {
                const double a0 = xa[ks * 4], a1 = xa[8 * XP + ks * 4];
                double b[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) b[c] = wb[ks * 4 * BD_CP + c * 8];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    bd_dmma(s1[0][c][0], s1[0][c][1], a0, b[c]);
                    bd_dmma(s1[1][c][0], s1[1][c][1], a1, b[c]);
                }
            }
        }
        // ---------------- epilogue: l += ln|S|^2, R = conj(S)/|S|^2 -> sR
#pragma unroll
        for (int m = 0; m < 2; ++m) {
            const int erow = (er * 2 + m) * 8 + lq;
            const bool valid = (t * BD_E + erow) < N;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const double sr = s1[m][c][0], si = s1[m][c][1];
                const double I = sr * sr + si * si;
                const double l = log(I);
                const double inv = 1.0 / I;
                double rr = sr * inv, ri = -si * inv;
                if (valid) { Lacc[c] += l; if (!(I > 0.0) || !isfinite(l)) badacc[c] += 1.0; }
                else { rr = 0.0; ri = 0.0; }
                *reinterpret_cast<double2 *>(sR + erow * BD_CP + (cg * 4 + c) * 8 + lr * 2) = make_double2(rr, ri);
            }
        }
        __syncthreads();
        // ---------------- GEMM2: Q[RB row blocks][CB column blocks] += X^T R over the tile's events
        {
            const double *xa = sX + lr * XP + (rg * RB) * 8 + lq;
            const double *rb = sR + lr * BD_CP + (cg2 * CB) * 8 + lq;
#pragma unroll 2
            for (int ks = 0; ks < BD_E / 4; ++ks) {
                double a[RB], b[CB];
#pragma unroll
                for (int i = 0; i < RB; ++i) a[i] = xa[ks * 4 * XP + i * 8];
#pragma unroll
                for (int j = 0; j < CB; ++j) b[j] = rb[ks * 4 * BD_CP + j * 8];
#pragma unroll
                for (int i = 0; i < RB; ++i)
#pragma unroll
                    for (int j = 0; j < CB; ++j) bd_dmma(q2[i][j][0], q2[i][j][1], a[i], b[j]);
            }
        }
    }
    __syncthreads();

    // ---- per-CTA partials -> fixed slot
    double *slot = scratch + (size_t)blockIdx.x * bd_slot_doubles(NB);
#pragma unroll
    for (int i = 0; i < RB; ++i)
#pragma unroll
        for (int j = 0; j < CB; ++j) {
            const int rbk = rg * RB + i, cbk = cg2 * CB + j;
            *reinterpret_cast<double2 *>(slot + ((size_t)rbk * 8 + cbk) * 64 + lq * 8 + lr * 2) = make_double2(q2[i][j][0], q2[i][j][1]);
        }
    // L and bad: reduce over the 8 event rows of the fragment (lane bits 2..4), then over the 4 event-row groups
#pragma unroll
    for (int c = 0; c < 4; ++c) {
#pragma unroll
        for (int m = 4; m < 32; m <<= 1) {
            Lacc[c] += __shfl_xor_sync(0xffffffffu, Lacc[c], m);
            badacc[c] += __shfl_xor_sync(0xffffffffu, badacc[c], m);
        }
        if (lq == 0) {
            const int kl = (cg * 4 + c) * 4 + lr;
            sL[er * 2 * BD_KC + kl] = Lacc[c];
            sL[er * 2 * BD_KC + BD_KC + kl] = badacc[c];
        }
    }
    __syncthreads();
    if (tid < 2 * BD_KC) {
        double v = 0.0;
#pragma unroll
        for (int g = 0; g < 4; ++g) v += sL[g * 2 * BD_KC + tid];
        slot[(size_t)NB * 8 * 64 + tid] = v;
    }
}

// One block per column: sums over the per-CTA slots in a fixed tree, Q -> T, then step A7 ->
// result record k0 + column.  1024 threads = 4 slot phases x 256 values (wave a, which of
// Q[2a][2k], Q[2a][2k+1], Q[2a+1][2k], Q[2a+1][2k+1]); warps 0 and 1 of phase 0 also add L and the
// non-finite count (lanes stride the slots, xor tree).
constexpr int BF_THREADS = 1024;
__global__ void __launch_bounds__(BF_THREADS)
k_batch_finalize(const double *__restrict__ scratch, int nslots, int NB, int n, const double *__restrict__ Vdev,
                 int k0, const double *__restrict__ M, double *__restrict__ results, int result_stride, bool eq2, double n_eq2,
                 unsigned long long *done_flags, unsigned long long seq)
{
    __shared__ double s_val[4][256];
    __shared__ double s_tot[2 + 2 * kFastWaves];
    __shared__ double sV[2 * kFastWaves];
    const int kl = blockIdx.x, k = k0 + kl, tid = threadIdx.x;
    const size_t sd = bd_slot_doubles(NB);
    const int v = tid & 255, ph = tid >> 8;
    {
        const int a = v >> 2, w = v & 3;
        double acc = 0.0;
        if (a < n) {
            const int rbk = a >> 2, cbk = kl >> 2, rr = ((2 * a) & 7) + (w >> 1), cc = ((2 * kl) & 7) + (w & 1);
            const double *src = scratch + ((size_t)rbk * 8 + cbk) * 64 + rr * 8 + cc;
            for (int s0 = ph; s0 < nslots; s0 += 16) {
                double x[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { const int sl = s0 + 4 * u; x[u] = (sl < nslots) ? __ldcg(src + (size_t)sl * sd) : 0.0; }
#pragma unroll
                for (int u = 0; u < 4; ++u) acc += x[u];
            }
        }
        s_val[ph][v] = acc;
    }
    if (tid < 64) {                                  // warp 0: L, warp 1: non-finite count
        const int which = tid >> 5, lane = tid & 31;
        double acc = 0.0;
        for (int s = lane; s < nslots; s += 32) acc += __ldcg(scratch + (size_t)s * sd + (size_t)NB * 8 * 64 + which * BD_KC + kl);
        acc = warp_sum(acc);
        if (lane == 0) s_tot[which] = acc;
    }
    __syncthreads();
    if (tid < n) {
        const int a = tid;
        double q[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) q[w] = ((s_val[0][4 * a + w] + s_val[1][4 * a + w]) + s_val[2][4 * a + w]) + s_val[3][4 * a + w];
        s_tot[2 + 2 * a] = q[0] - q[3];              // Re T = Q[2a][2k] - Q[2a+1][2k+1]
        s_tot[3 + 2 * a] = q[1] + q[2];              // Im T = Q[2a][2k+1] + Q[2a+1][2k]
        sV[2 * a] = Vdev[((size_t)k * n + a) * 2];
        sV[2 * a + 1] = Vdev[((size_t)k * n + a) * 2 + 1];
    }
    __syncthreads();
    assemble_from_totals(s_tot, sV, M, results + (size_t)k * result_stride, n, eq2, n_eq2, done_flags + k, seq);
}

template <typename ST, int NB, bool ALIGNED>
static pwa_status launch_bd(pwa_ctx *ctx, int K)
{
    using C = BatchCfg<NB>;
    auto kern = k_batch_dmma<ST, NB, ALIGNED>;
    PWA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    const long long N = ctx->data.n_events;
    const long long ntiles = (N + BD_E - 1) / BD_E;
    long long grid = ctx->sm_count;
    if (grid > ntiles) grid = ntiles;
    if (grid < 1) grid = 1;
    pwa_status s = ensure_scratch(ctx, sizeof(double) * (size_t)grid * bd_slot_doubles(NB));
    if (s != PWA_OK) return s;
    for (int k0 = 0; k0 < K; k0 += BD_KC) {
        kern<<<(unsigned)grid, BD_THREADS, C::SMEM, ctx->stream>>>(ctx->data.amps, N, ctx->n, ctx->d_V, K, k0, ctx->d_scratch);
        ctx->launches++;
        PWA_CUDA(ctx, cudaGetLastError());
        const int cols = (K - k0 < BD_KC) ? (K - k0) : BD_KC;
        k_batch_finalize<<<cols, BF_THREADS, 0, ctx->stream>>>(ctx->d_scratch, (int)grid, NB, ctx->n, ctx->d_V, k0, ctx->d_M,
                                                        ctx->dev_result, result_stride(ctx->n),
                                                        ctx->opt_likelihood == 1, eq2_n_data(ctx),
                                                        ctx->dev_flags, ctx->seq);
        ctx->launches++;
        PWA_CUDA(ctx, cudaGetLastError());
    }
    return PWA_OK;
}

template <typename ST, bool ALIGNED>
static pwa_status dispatch_bd(pwa_ctx *ctx, int K)
{
    const int D = 2 * ctx->n;
    if (D <= 8)  return launch_bd<ST, 1, ALIGNED>(ctx, K);
    if (D <= 16) return launch_bd<ST, 2, ALIGNED>(ctx, K);
    if (D <= 32) return launch_bd<ST, 4, ALIGNED>(ctx, K);
    if (D <= 64) return launch_bd<ST, 8, ALIGNED>(ctx, K);
    return launch_bd<ST, 16, ALIGNED>(ctx, K);
}

// Handles constant-resonance samples with n <= 64 and K >= 8 (below that K single passes of the
// streaming kernel read fewer bytes than one padded 32-column GEMM pass costs in flops).
pwa_status launch_batch_dmma(pwa_ctx *ctx, int K, bool *handled)
{
    *handled = false;
    const int n = ctx->n;
    if (ctx->data.factored || n > kMaxFastWaves || ctx->data.n_events == 0) return PWA_OK;
    if (K < 8 && ctx->opt_batch != 1) return PWA_OK;
    const bool f32 = ctx->storage == PWA_F32;
    const bool pow2 = (n & (n - 1)) == 0 && n >= 4;
    const bool aligned = pow2 && ((uintptr_t)ctx->data.amps & 15u) == 0;
    pwa_status s;
    if (aligned) s = f32 ? dispatch_bd<float, true>(ctx, K) : dispatch_bd<double, true>(ctx, K);
    else         s = f32 ? dispatch_bd<float, false>(ctx, K) : dispatch_bd<double, false>(ctx, K);
    if (s != PWA_OK) return s;
    *handled = true;
    return PWA_OK;
}

}  // namespace pwa
