// norm_dmma.cu — step A6 on the FP64 tensor cores:
//     M_ab = (1/N_gen) sum_j conj(B_ja) B_jb          (P:41 inner bracket, reading C1)
// B200's tcgen05.mma has no f64 kind, so the fp64 contraction is issued as warp-level
// mma.sync.m8n8k4.f64 (DMMA).  Real embedding: the interleaved (re, im) buffer IS the real
// matrix X = B_r [N_acc x D], D = 2n, and P = X^T X (D x D, symmetric) gives
//     Re M_ab = P[2a][2b] + P[2a+1][2b+1],   Im M_ab = P[2a][2b+1] - P[2a+1][2b]
// so no de-interleave pass is needed.  The long dimension (events) is the contraction index k.
//
// Fragment identity used here: for an 8-column block cb and a quad of 4 events e0..e0+3, the value
//     F[cb](lane) = X[e0 + lane%4][8 cb + lane/4]
// is at the same time the A operand (8x4, row) of row-block cb and the B operand (4x8, col) of
// column-block cb, so a warp loads D/8 fragments per quad from the shared-memory tile and issues
// one DMMA per block pair (i <= j) it owns.  Accumulators (8x8 per pair, 2 doubles per lane) stay
// in registers for the CTA's whole event range (split-K); every (CTA, warp group) writes its
// partial upper-triangle blocks to a fixed slot and k_norm_dmma_finalize sums the slots in slot
// order (bitwise reproducible), scales by 1/N_gen and writes both triangles (exactly Hermitian).
//
// Tile rows are padded to DP = D + 4 doubles (DP mod 16 in {4, 12}) so that the fragment load
// LDS.64 is bank-conflict free.  fp32-stored amplitudes are widened when the tile is written
// (exact, C16).  Factored mode (A1): the tile producer recomputes BW(m_j; M_r, G_r) * Z_js.
#include "pwa_internal.h"
#include "factored.cuh"

namespace pwa {

__device__ __forceinline__ void dmma_884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ uint4 ldg_stream16(const uint4 *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

enum FillMode { FILL_STAGED = 0, FILL_ELEMENT = 1, FILL_FACTORED = 2 };

constexpr int npairs_of(int nb) { return nb * (nb + 1) / 2; }

// One quad (4 events) of the tile: load the fragments, issue this warp's DMMAs.
template <int NB, int SPLIT, int S, int PPW>
__device__ __forceinline__ void quad_mma(const double *__restrict__ tq, int DP, int lane, double (&acc)[PPW][2])
{
    double f[NB];
    const double *src = tq + (lane & 3) * DP + (lane >> 2);
#pragma unroll
    for (int cb = 0; cb < NB; ++cb) f[cb] = src[cb * 8];
    int p = 0;
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
        for (int j = i; j < NB; ++j) {
            if (p % SPLIT == S) dmma_884(acc[p / SPLIT][0], acc[p / SPLIT][1], f[i], f[j]);
            ++p;
        }
}

template <typename ST, int NB, int SPLIT, int MODE, int THREADS, int ET>
struct NormCfg {
    static constexpr int D = NB * 8, DP = D + 4, W = THREADS / 32, NG = W / SPLIT, QPT = ET / 4;
    static constexpr int NPAIRS = npairs_of(NB), PPW = (NPAIRS + SPLIT - 1) / SPLIT;
    static constexpr int CH = 16 / (int)sizeof(ST);          // elements per 16-byte chunk
    static constexpr int RC = D / CH;                          // chunks per (unpadded) row
    static constexpr int CPT = (ET * RC + THREADS - 1) / THREADS;
    static constexpr size_t SMEM = sizeof(double) * 2 * ET * DP;
};

template <typename ST, int NB, int SPLIT, int MODE, int THREADS, int ET, int S>
__device__ __forceinline__ void norm_body(const void *__restrict__ Bv, long long N, int n, const FactArgs &f,
                                          double *__restrict__ scratch, double *smem)
{
    using C = NormCfg<ST, NB, SPLIT, MODE, THREADS, ET>;
    constexpr int D = C::D, DP = C::DP, NG = C::NG, QPT = C::QPT, PPW = C::PPW, NPAIRS = C::NPAIRS;
    constexpr int CH = C::CH, RC = C::RC, CPT = C::CPT;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, group = warp / SPLIT;
    double *buf[2] = {smem, smem + ET * DP};

    double acc[PPW][2];
#pragma unroll
    for (int p = 0; p < PPW; ++p) { acc[p][0] = 0.0; acc[p][1] = 0.0; }

    const long long ntiles = (N + ET - 1) / ET;
    uint4 stage[CPT];   // FILL_STAGED only (dead otherwise)

    auto load_tile = [&](long long t) {                       // FILL_STAGED: global -> registers
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            const int idx = tid + c * THREADS;
            const int e = idx / RC, ch = idx % RC;
            const long long ev = t * ET + e;
            if (idx < ET * RC && ev < N) stage[c] = ldg_stream16(reinterpret_cast<const uint4 *>(Bv) + ev * RC + ch);
            else                         stage[c] = make_uint4(0u, 0u, 0u, 0u);
        }
    };
    auto store_tile = [&](double *dst) {                      // FILL_STAGED: registers -> smem (fp64)
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            const int idx = tid + c * THREADS;
            if (idx >= ET * RC) continue;
            const int e = idx / RC, ch = idx % RC;
            double *d = dst + e * DP + ch * CH;
            if (sizeof(ST) == 8) {
                *reinterpret_cast<double2 *>(d) = make_double2(__hiloint2double((int)stage[c].y, (int)stage[c].x),
                                                               __hiloint2double((int)stage[c].w, (int)stage[c].z));
            } else {
                *reinterpret_cast<double2 *>(d) = make_double2((double)__uint_as_float(stage[c].x), (double)__uint_as_float(stage[c].y));
                *reinterpret_cast<double2 *>(d + 2) = make_double2((double)__uint_as_float(stage[c].z), (double)__uint_as_float(stage[c].w));
            }
        }
    };
    auto fill_tile = [&](double *dst, long long t) {          // FILL_ELEMENT / FILL_FACTORED: direct
        if constexpr (MODE == FILL_ELEMENT) {
            const ST *B = reinterpret_cast<const ST *>(Bv);
            const int d2 = 2 * n;
            for (int idx = tid; idx < ET * D; idx += THREADS) {
                const int e = idx / D, c = idx % D;
                const long long ev = t * ET + e;
                dst[e * DP + c] = (ev < N && c < d2) ? (double)B[ev * d2 + c] : 0.0;
            }
        } else {
            const int nres = f.n_res;
            for (int idx = tid; idx < ET * nres; idx += THREADS) {
                const int e = idx / nres, r = idx % nres;
                const long long ev = t * ET + e;
                const bool valid = ev < N;
                double2 bw = make_double2(0.0, 0.0);
                if (valid) { const double m = f.mass[ev]; bw = bw_eval(m * m, f.rp.m2[r], f.rp.mg[r]); }
                for (int s = 0; s < f.n_ang; ++s) {
                    const int w = f.wave_of_pair[r * kMaxAng + s];
                    if (w < 0) continue;
                    double2 a = make_double2(0.0, 0.0);
                    if (valid) {
                        const double2 z = load_ang<ST>(f.ang, ev, f.n_ang, s);
                        a = make_double2(bw.x * z.x - bw.y * z.y, bw.x * z.y + bw.y * z.x);
                    }
                    *reinterpret_cast<double2 *>(dst + e * DP + 2 * w) = a;
                }
            }
        }
    };
    auto compute = [&](const double *src) {
#pragma unroll 1
        for (int q = group; q < QPT; q += NG) quad_mma<NB, SPLIT, S, PPW>(src + q * 4 * DP, DP, lane, acc);
    };

    if (MODE == FILL_FACTORED) {                              // padded / unmapped columns stay zero
        for (int idx = tid; idx < 2 * ET * DP; idx += THREADS) smem[idx] = 0.0;
        __syncthreads();
    }
    long long t = blockIdx.x;
    int cur = 0;
    if (t < ntiles) {
        if constexpr (MODE == FILL_STAGED) { load_tile(t); store_tile(buf[0]); }
        else fill_tile(buf[0], t);
    }
    __syncthreads();
    for (; t < ntiles; t += gridDim.x) {
        const long long nxt = t + gridDim.x;
        if constexpr (MODE == FILL_STAGED) {
            if (nxt < ntiles) load_tile(nxt);
            compute(buf[cur]);
            if (nxt < ntiles) store_tile(buf[cur ^ 1]);
        } else {
            compute(buf[cur]);
            if (nxt < ntiles) fill_tile(buf[cur ^ 1], nxt);
        }
        __syncthreads();
        cur ^= 1;
    }
    // partial blocks of this (CTA, group) -> fixed slot, [pair][8][8] doubles
    const size_t slot = (size_t)blockIdx.x * NG + group;
    double *dst = scratch + slot * (size_t)NPAIRS * 64 + (lane >> 2) * 8 + (lane & 3) * 2;
#pragma unroll
    for (int pl = 0; pl < PPW; ++pl) {
        const int p = pl * SPLIT + S;
        if (p < NPAIRS) *reinterpret_cast<double2 *>(dst + (size_t)p * 64) = make_double2(acc[pl][0], acc[pl][1]);
    }
}

template <typename ST, int NB, int SPLIT, int MODE, int THREADS, int MINB, int ET>
__global__ void __launch_bounds__(THREADS, MINB)
k_norm_dmma(const void *__restrict__ Bv, long long N, int n, FactArgs f, double *__restrict__ scratch)
{
    extern __shared__ double nd_smem[];
    const int S = (threadIdx.x >> 5) % SPLIT;
    if (SPLIT == 1) { norm_body<ST, NB, SPLIT, MODE, THREADS, ET, 0>(Bv, N, n, f, scratch, nd_smem); return; }
    switch (S) {        // warp-uniform: each sub-id owns a compile-time list of block pairs
    case 0: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, 0>(Bv, N, n, f, scratch, nd_smem); break;
    case 1: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, (SPLIT > 1 ? 1 : 0)>(Bv, N, n, f, scratch, nd_smem); break;
    case 2: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, (SPLIT > 2 ? 2 : 0)>(Bv, N, n, f, scratch, nd_smem); break;
    default: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, (SPLIT > 3 ? 3 : 0)>(Bv, N, n, f, scratch, nd_smem); break;
    }
}

// One warp per complex entry (a <= b): lanes stride over the slots, fixed xor tree.
__global__ void __launch_bounds__(256)
k_norm_dmma_finalize(const double *__restrict__ scratch, int nslots, int n, int NB, double inv_ngen,
                     double *__restrict__ M)
{
    const int lane = threadIdx.x & 31;
    const long long wid = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nent = (long long)n * (n + 1) / 2;
    if (wid >= nent) return;
    int a = 0; long long q = wid;
    while (q >= n - a) { q -= n - a; ++a; }
    const int b = a + (int)q;
    const int i = a >> 2, j = b >> 2;
    const int p = i * NB - i * (i - 1) / 2 + (j - i);
    const int rr = (2 * a) & 7, cc = (2 * b) & 7;
    const int npairs = NB * (NB + 1) / 2;
    double p00 = 0.0, p11 = 0.0, p01 = 0.0, p10 = 0.0;
    for (int s = lane; s < nslots; s += 32) {
        const double *blk = scratch + ((size_t)s * npairs + p) * 64;
        p00 += blk[rr * 8 + cc];       p01 += blk[rr * 8 + cc + 1];
        p10 += blk[(rr + 1) * 8 + cc]; p11 += blk[(rr + 1) * 8 + cc + 1];
    }
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        p00 += __shfl_xor_sync(0xffffffffu, p00, m); p01 += __shfl_xor_sync(0xffffffffu, p01, m);
        p10 += __shfl_xor_sync(0xffffffffu, p10, m); p11 += __shfl_xor_sync(0xffffffffu, p11, m);
    }
    if (lane == 0) {
        const double re = (p00 + p11) * inv_ngen;
        const double im = (a == b) ? 0.0 : (p01 - p10) * inv_ngen;      // |B_ja|^2 is real
        M[((size_t)a * n + b) * 2] = re;  M[((size_t)a * n + b) * 2 + 1] = im;
        if (a != b) { M[((size_t)b * n + a) * 2] = re;  M[((size_t)b * n + a) * 2 + 1] = -im; }
    }
}

template <typename ST, int NB, int SPLIT, int MODE, int MINB, int ET>
static pwa_status launch_nd(pwa_ctx *ctx, const FactArgs &fargs)
{
    constexpr int THREADS = 256;
    using C = NormCfg<ST, NB, SPLIT, MODE, THREADS, ET>;
    auto kern = k_norm_dmma<ST, NB, SPLIT, MODE, THREADS, MINB, ET>;
    PWA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
    int occ = 0;
    PWA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, C::SMEM));
    if (occ < 1) occ = 1;
    const long long N = ctx->mc.n_events;
    const long long ntiles = (N + ET - 1) / ET;
    long long grid = (long long)ctx->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    if (grid < 1) grid = 1;
    const int nslots = (int)grid * C::NG;
    pwa_status s = ensure_scratch(ctx, sizeof(double) * (size_t)nslots * C::NPAIRS * 64);
    if (s != PWA_OK) return s;
    kern<<<(unsigned)grid, THREADS, C::SMEM, ctx->stream>>>(ctx->mc.factored ? nullptr : ctx->mc.amps, N, ctx->n, fargs, ctx->d_scratch);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    const long long nent = (long long)ctx->n * (ctx->n + 1) / 2;
    const int fblocks = (int)((nent * 32 + 255) / 256);
    k_norm_dmma_finalize<<<fblocks, 256, 0, ctx->stream>>>(ctx->d_scratch, nslots, ctx->n, NB,
                                                          1.0 / (double)ctx->mc.n_gen, ctx->d_M);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

template <typename ST, int MODE>
static pwa_status dispatch_nd(pwa_ctx *ctx, const FactArgs &fargs)
{
    const int D = 2 * ctx->n;
    //                                   NB SPLIT      MINB ET
    if (D <= 8)   return launch_nd<ST, 1,  1, MODE, 2, 128>(ctx, fargs);
    if (D <= 16)  return launch_nd<ST, 2,  1, MODE, 2, 128>(ctx, fargs);
    if (D <= 32)  return launch_nd<ST, 4,  1, MODE, 2, 128>(ctx, fargs);
    if (D <= 64)  return launch_nd<ST, 8,  2, MODE, 2, 64>(ctx, fargs);
    return launch_nd<ST, 16, 4, MODE, 1, 32>(ctx, fargs);
}

pwa_status launch_norm_dmma(pwa_ctx *ctx, bool *handled)
{
    *handled = false;
    const int n = ctx->n;
    if (n > kMaxFastWaves) return PWA_OK;                      // generic CUDA-core kernel handles it
    FactArgs fargs;
    const bool fact = ctx->mc.factored;
    if (fact) {
        pwa_status s = fill_fact_args(ctx, ctx->mc, &fargs);
        if (s != PWA_OK) return s;
    } else {
        memset(&fargs, 0, sizeof(fargs));
    }
    const bool f32 = ctx->storage == PWA_F32;
    const bool pow2 = (n & (n - 1)) == 0 && n >= 4;            // rows are whole 16-byte chunks, D = 2n
    const bool aligned = ((uintptr_t)ctx->mc.amps & 15u) == 0;
    pwa_status s;
    if (fact)                 s = f32 ? dispatch_nd<float, FILL_FACTORED>(ctx, fargs) : dispatch_nd<double, FILL_FACTORED>(ctx, fargs);
    else if (pow2 && aligned) s = f32 ? dispatch_nd<float, FILL_STAGED>(ctx, fargs)   : dispatch_nd<double, FILL_STAGED>(ctx, fargs);
    else                      s = f32 ? dispatch_nd<float, FILL_ELEMENT>(ctx, fargs)  : dispatch_nd<double, FILL_ELEMENT>(ctx, fargs);
    if (s != PWA_OK) return s;
    *handled = true;
    return PWA_OK;
}

}  // namespace pwa
