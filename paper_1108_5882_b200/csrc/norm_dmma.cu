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
// in registers for the CTA's whole event range (split-K); the CTA's warp groups are summed in group
// order, every CTA writes its partial upper-triangle blocks to a fixed slot and k_norm_dmma_finalize
// sums the slots in a fixed tree (bitwise reproducible), scales by 1/N_gen and writes both
// triangles (exactly Hermitian).
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

// Weighted quad (NEXT-3): the event weight w_e sits in the first padding column of the tile row
// (tile[e][D]); the A-operand fragment is scaled by it, sum_e w_e X[e][p] X[e][q].
template <int NB, int SPLIT, int S, int PPW>
__device__ __forceinline__ void quad_mma_w(const double *__restrict__ tq, int DP, int lane, double (&acc)[PPW][2])
{
    double f[NB], fw[NB];
    const double *src = tq + (lane & 3) * DP + (lane >> 2);
    const double w = tq[(lane & 3) * DP + NB * 8];
#pragma unroll
    for (int cb = 0; cb < NB; ++cb) { f[cb] = src[cb * 8]; fw[cb] = f[cb] * w; }
    int p = 0;
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
        for (int j = i; j < NB; ++j) {
            if (p % SPLIT == S) dmma_884(acc[p / SPLIT][0], acc[p / SPLIT][1], fw[i], f[j]);
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
    static constexpr size_t SMEM = sizeof(double) * (2 * ET * DP > NPAIRS * 64 ? 2 * ET * DP : NPAIRS * 64);   // tiles, then the CTA partial
};

template <typename ST, int NB, int SPLIT, int MODE, int THREADS, int ET, int S, int NANG, bool EXTRA>
__device__ __forceinline__ void norm_body(const void *__restrict__ Bv, long long N, int n, const FactArgs &f,
                                          double *__restrict__ scratch, double *smem, const double *__restrict__ Vs,
                                          const double *__restrict__ Wt)
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
    // FILL_FACTORED: thread -> (event e = tid % ET, resonance subset part, part + TPE, ...); the mass
    // and the angular factors of the NEXT tile are fetched into registers before the DMMAs of the
    // current one, so their latency is hidden (the event's TPE threads load the same 8 + 16 n_ang bytes)
    constexpr int TPE = THREADS / ET;
    static_assert(THREADS % ET == 0, "whole threads per event");
    double pm = 0.0;
    double2 pz[NANG];
    auto fact_load = [&](long long t) {
        const long long ev = t * ET + (tid % ET);
        const bool valid = ev < N;
        pm = valid ? __ldg(f.mass + ev) : 0.0;
#pragma unroll
        for (int s = 0; s < NANG; ++s)
            pz[s] = (valid && s < f.n_ang) ? load_ang<ST>(f.ang, ev, f.n_ang, s) : make_double2(0.0, 0.0);
    };
    auto fact_store = [&](double *dst) {                       // A1: BW(m_j; M_r, G_r) * Z_js -> tile (fp64)
        double *row = dst + (tid % ET) * DP;
        const double m2 = pm * pm;
        for (int r = tid / ET; r < f.n_res; r += TPE) {        // warp-uniform r: parameters come from the constant bank
            const double2 bw = bw_eval_fast(m2, f.rp.m2[r], f.rp.mg[r]);
#pragma unroll
            for (int s = 0; s < NANG; ++s) {
                const int w = f.wave_of_pair[r * kMaxAng + s];
                if (w >= 0)
                    *reinterpret_cast<double2 *>(row + 2 * w) =
                        make_double2(bw.x * pz[s].x - bw.y * pz[s].y, bw.x * pz[s].y + bw.y * pz[s].x);
            }
        }
    };

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
        }
    };
    // Fumili mode (Vs != nullptr): every row of the tile is replaced by
    // t_i = A_i / S_i, S_i = sum_a V_a A_ia, so that the Gram matrix becomes sum_i (Re t, Im t)(Re t, Im t)^T.
    // TPS adjacent lanes share an event (xor-shuffle sum of the partial S); rows past N stay zero.
    auto scale_tile = [&](double *tile, long long t) {
        constexpr int TPS = THREADS / ET;
        const int e = tid / TPS, part = tid % TPS;
        double *row = tile + e * DP;
        double sr = 0.0, si = 0.0;
        for (int a = part; a < n; a += TPS) {
            const double2 x = *reinterpret_cast<const double2 *>(row + 2 * a);
            const double vr = __ldg(Vs + 2 * a), vi = __ldg(Vs + 2 * a + 1);
            sr = fma(vr, x.x, sr); sr = fma(-vi, x.y, sr);
            si = fma(vr, x.y, si); si = fma(vi, x.x, si);
        }
#pragma unroll
        for (int m = 1; m < TPS; m <<= 1) { sr += __shfl_xor_sync(0xffffffffu, sr, m); si += __shfl_xor_sync(0xffffffffu, si, m); }
        if (t * ET + e < N) {
            const double I = sr * sr + si * si, inv = 1.0 / I, rr = sr * inv, ri = -si * inv;      // r = 1 / S = conj(S) / I
            for (int a = part; a < n; a += TPS) {
                const double2 x = *reinterpret_cast<const double2 *>(row + 2 * a);
                *reinterpret_cast<double2 *>(row + 2 * a) = make_double2(x.x * rr - x.y * ri, x.x * ri + x.y * rr);
            }
        }
    };
    auto compute = [&](const double *src) {
        if (EXTRA && Wt != nullptr) {
#pragma unroll 1
            for (int q = group; q < QPT; q += NG) quad_mma_w<NB, SPLIT, S, PPW>(src + q * 4 * DP, DP, lane, acc);
        } else {
#pragma unroll 1
            for (int q = group; q < QPT; q += NG) quad_mma<NB, SPLIT, S, PPW>(src + q * 4 * DP, DP, lane, acc);
        }
    };
    auto fill_w = [&](double *dst, long long t) {             // event weights -> padding column D of the tile
        if (!EXTRA || Wt == nullptr) return;
        for (int e = tid; e < ET; e += THREADS) {
            const long long ev = t * ET + e;
            dst[e * DP + D] = ev < N ? __ldg(Wt + ev) : 0.0;
        }
    };

    if (MODE == FILL_FACTORED) {                              // padded / unmapped columns stay zero
        for (int idx = tid; idx < 2 * ET * DP; idx += THREADS) smem[idx] = 0.0;
        __syncthreads();
    }
    long long t = blockIdx.x;
    int cur = 0;
    if (t < ntiles) {
        if constexpr (MODE == FILL_STAGED) { load_tile(t); store_tile(buf[0]); }
        else if constexpr (MODE == FILL_FACTORED) { fact_load(t); fact_store(buf[0]); }
        else fill_tile(buf[0], t);
        fill_w(buf[0], t);
    }
    __syncthreads();
    for (; t < ntiles; t += gridDim.x) {
        const long long nxt = t + gridDim.x;
        if (EXTRA && Vs != nullptr) { scale_tile(buf[cur], t); __syncthreads(); }
        if constexpr (MODE == FILL_STAGED) {
            if (nxt < ntiles) load_tile(nxt);
            compute(buf[cur]);
            if (nxt < ntiles) store_tile(buf[cur ^ 1]);
        } else if constexpr (MODE == FILL_FACTORED) {
            if (nxt < ntiles) fact_load(nxt);
            compute(buf[cur]);
            if (nxt < ntiles) fact_store(buf[cur ^ 1]);
        } else {
            compute(buf[cur]);
            if (nxt < ntiles) fill_tile(buf[cur ^ 1], nxt);
        }
        if (nxt < ntiles) fill_w(buf[cur ^ 1], nxt);
        __syncthreads();
        cur ^= 1;
    }
    // the CTA's groups are summed in group order in shared memory (the tile buffers are free after
    // the loop's last barrier), then ONE partial per CTA goes to its fixed slot, [pair][8][8] doubles
    double *red = smem;
    for (int g = 0; g < NG; ++g) {
        if (group == g) {
            double *dst = red + (lane >> 2) * 8 + (lane & 3) * 2;
#pragma unroll
            for (int pl = 0; pl < PPW; ++pl) {
                const int p = pl * SPLIT + S;
                if (p < NPAIRS) {
                    double2 v = make_double2(acc[pl][0], acc[pl][1]);
                    if (g > 0) { const double2 o = *reinterpret_cast<double2 *>(dst + p * 64); v.x += o.x; v.y += o.y; }
                    *reinterpret_cast<double2 *>(dst + p * 64) = v;
                }
            }
        }
        __syncthreads();
    }
    double *slot = scratch + (size_t)blockIdx.x * NPAIRS * 64;
    for (int idx = tid; idx < NPAIRS * 64; idx += THREADS) slot[idx] = red[idx];
}

// EXTRA = true adds the row-scaling (Fumili, Vs) and event-weight (Wt) passes; the plain M build
// (EXTRA = false) compiles to the same code as before they existed.
template <typename ST, int NB, int SPLIT, int MODE, int THREADS, int MINB, int ET, int NANG, bool EXTRA>
__global__ void __launch_bounds__(THREADS, MINB)
k_norm_dmma(const void *__restrict__ Bv, long long N, int n, FactArgs f, double *__restrict__ scratch,
            const double *__restrict__ Vs, const double *__restrict__ Wt)
{
    extern __shared__ double nd_smem[];
    const int S = (threadIdx.x >> 5) % SPLIT;
    if (SPLIT == 1) { norm_body<ST, NB, SPLIT, MODE, THREADS, ET, 0, NANG, EXTRA>(Bv, N, n, f, scratch, nd_smem, Vs, Wt); return; }
    switch (S) {        // warp-uniform: each sub-id owns a compile-time list of block pairs
    case 0: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, 0, NANG, EXTRA>(Bv, N, n, f, scratch, nd_smem, Vs, Wt); break;
    case 1: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, (SPLIT > 1 ? 1 : 0), NANG, EXTRA>(Bv, N, n, f, scratch, nd_smem, Vs, Wt); break;
    case 2: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, (SPLIT > 2 ? 2 : 0), NANG, EXTRA>(Bv, N, n, f, scratch, nd_smem, Vs, Wt); break;
    default: norm_body<ST, NB, SPLIT, MODE, THREADS, ET, (SPLIT > 3 ? 3 : 0), NANG, EXTRA>(Bv, N, n, f, scratch, nd_smem, Vs, Wt); break;
    }
}

// Final sum over the per-CTA slots and P -> M.  One block per (block pair p, row pair k): its 16
// elements are rows 2k, 2k+1 of the 8 x 8 block = one wave a (re, im rows) against the 4 waves of
// the column block.  256 threads = 16 elements x 16 slot phases: thread (el, ph) adds slots ph,
// ph + 16, ... (coalesced 128-byte reads, independent loads), the phases are then added in phase
// order: a fixed tree, bitwise reproducible for a fixed grid.
__global__ void __launch_bounds__(256)
k_norm_dmma_finalize(const double *__restrict__ scratch, int nslots, int n, int NB, double inv_ngen,
                     double *__restrict__ M)
{
    __shared__ double s_ph[16][17];
    __shared__ double s_tot[16];
    const int p = blockIdx.x >> 2, k = blockIdx.x & 3;
    const int el = threadIdx.x & 15, ph = threadIdx.x >> 4;
    const size_t stride = (size_t)NB * (NB + 1) / 2 * 64;
    const double *src = scratch + (size_t)p * 64 + k * 16 + el;
    double acc = 0.0;
    for (int s0 = ph; s0 < nslots; s0 += 64) {
        double x[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int sl = s0 + 16 * u; x[u] = (sl < nslots) ? __ldcg(src + (size_t)sl * stride) : 0.0; }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc += x[u];
    }
    s_ph[ph][el] = acc;
    __syncthreads();
    if (threadIdx.x < 16) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < 16; ++q) t += s_ph[q][threadIdx.x];
        s_tot[threadIdx.x] = t;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        int i = 0, q = p;
        while (q >= NB - i) { q -= NB - i; ++i; }
        const int j = i + q;
        const int a = 4 * i + k, b = 4 * j + (int)threadIdx.x, cc = 2 * (int)threadIdx.x;
        if (a < n && b < n && a <= b) {
            const double re = (s_tot[cc] + s_tot[8 + cc + 1]) * inv_ngen;                       // P[2a][2b] + P[2a+1][2b+1]
            const double im = (a == b) ? 0.0 : (s_tot[cc + 1] - s_tot[8 + cc]) * inv_ngen;      // P[2a][2b+1] - P[2a+1][2b]
            M[((size_t)a * n + b) * 2] = re;  M[((size_t)a * n + b) * 2 + 1] = im;
            if (a != b) { M[((size_t)b * n + a) * 2] = re;  M[((size_t)b * n + a) * 2 + 1] = -im; }
        }
    }
}

// Fumili finalize: H[p][q] = +-4 P[p][q] (+ Hess(Norm) from M when M != nullptr),
// P = sum over slots of the real Gram of t_i = A_i / S_i; sign - when exactly one of p, q is an
// imaginary-part index (u_i = (2 Re t, -2 Im t)).  Thread per element p <= q, mirrored: exactly symmetric.
__global__ void __launch_bounds__(256)
k_fumili_finalize(const double *__restrict__ scratch, int nslots, int n, int NB, const double *__restrict__ M,
                  double *__restrict__ H)
{
    const int D = 2 * n, idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= D * D) return;
    const int p = idx / D, q = idx % D;
    if (p > q) return;
    const int i = p >> 3, j = q >> 3;                      // block pair (i <= j)
    const int pair = i * NB - i * (i - 1) / 2 + (j - i);
    const size_t stride = (size_t)NB * (NB + 1) / 2 * 64;
    const double *src = scratch + (size_t)pair * 64 + (p & 7) * 8 + (q & 7);
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int s = 0;
    for (; s + 4 <= nslots; s += 4) {
        a0 += __ldcg(src + (size_t)s * stride);       a1 += __ldcg(src + (size_t)(s + 1) * stride);
        a2 += __ldcg(src + (size_t)(s + 2) * stride); a3 += __ldcg(src + (size_t)(s + 3) * stride);
    }
    for (; s < nslots; ++s) a0 += __ldcg(src + (size_t)s * stride);
    double h = (((p ^ q) & 1) ? -4.0 : 4.0) * ((a0 + a1) + (a2 + a3));
    if (M != nullptr) {
        const int a = p >> 1, b = q >> 1;
        const double mr = M[((size_t)a * n + b) * 2], mi = M[((size_t)a * n + b) * 2 + 1];
        // Hess(Norm) = 2 [[Re M, -Im M], [Im M, Re M]] on the (x_a, y_a) x (x_b, y_b) block
        h += ((p & 1) == (q & 1)) ? 2.0 * mr : ((p & 1) ? 2.0 * mi : -2.0 * mi);
    }
    H[(size_t)p * D + q] = h;
    H[(size_t)q * D + p] = h;
}

// smp: the sample whose Gram matrix is formed (MC for M; DATA for the Fumili matrix, with Vs = V on
// the device and H_out = the [2n][2n] device output, use_M = add Hess(Norm)).
struct GramJob { const Sample *smp; const double *Vs; double *H_out; bool use_M; };

template <typename ST, int NB, int SPLIT, int MODE, int MINB, int ET, int NANG>
static pwa_status launch_nd(pwa_ctx *ctx, const FactArgs &fargs, const GramJob &job)
{
    constexpr int THREADS = 256;
    using C = NormCfg<ST, NB, SPLIT, MODE, THREADS, ET>;
    const bool extra = job.Vs != nullptr || job.smp->weights != nullptr;
    auto kern = extra ? k_norm_dmma<ST, NB, SPLIT, MODE, THREADS, MINB, ET, NANG, true>
                      : k_norm_dmma<ST, NB, SPLIT, MODE, THREADS, MINB, ET, NANG, false>;
    static int s_occ2[2][64] = {{0}};                           // per instantiation and device
    int &occ = s_occ2[extra ? 1 : 0][ctx->device & 63];
    if (occ == 0) {
        PWA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        int o = 0;
        PWA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kern, THREADS, C::SMEM));
        occ = o < 1 ? 1 : o;
    }
    const long long N = job.smp->n_events;
    const long long ntiles = (N + ET - 1) / ET;
    long long grid = (long long)ctx->sm_count * occ;
    if (grid > ntiles) grid = ntiles;
    if (grid < 1) grid = 1;
    const int nslots = (int)grid;
    pwa_status s = ensure_scratch(ctx, sizeof(double) * (size_t)nslots * C::NPAIRS * 64);
    if (s != PWA_OK) return s;
    kern<<<(unsigned)grid, THREADS, C::SMEM, ctx->stream>>>(job.smp->factored ? nullptr : job.smp->amps, N, ctx->n, fargs, ctx->d_scratch, job.Vs, job.smp->weights);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    if (job.Vs != nullptr) {
        const int D2 = 4 * ctx->n * ctx->n;
        k_fumili_finalize<<<(D2 + 255) / 256, 256, 0, ctx->stream>>>(ctx->d_scratch, nslots, ctx->n, NB,
                                                                       job.use_M ? ctx->d_M : nullptr, job.H_out);
        ctx->launches++;
        PWA_CUDA(ctx, cudaGetLastError());
        return PWA_OK;
    }
    k_norm_dmma_finalize<<<C::NPAIRS * 4, 256, 0, ctx->stream>>>(ctx->d_scratch, nslots, ctx->n, NB,
                                                                 1.0 / (double)ctx->mc.n_gen, ctx->d_M);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

template <typename ST, int MODE, int NANG>
static pwa_status dispatch_nd(pwa_ctx *ctx, const FactArgs &fargs, const GramJob &job)
{
    const int D = 2 * ctx->n;
    //                                   NB SPLIT      MINB ET
    if (D <= 8)   return launch_nd<ST, 1,  1, MODE, 2, 128, NANG>(ctx, fargs, job);
    if (D <= 16)  return launch_nd<ST, 2,  1, MODE, 2, 128, NANG>(ctx, fargs, job);
    if (D <= 32)  return launch_nd<ST, 4,  1, MODE, 2, 128, NANG>(ctx, fargs, job);
    if (D <= 64)  return launch_nd<ST, 8,  2, MODE, 2, 64, NANG>(ctx, fargs, job);
    return launch_nd<ST, 16, 4, MODE, 1, 64, NANG>(ctx, fargs, job);
}

static pwa_status run_gram(pwa_ctx *ctx, const GramJob &job, bool *handled)
{
    *handled = false;
    const int n = ctx->n;
    const Sample &smp = *job.smp;
    if (n > kMaxFastWaves) return PWA_OK;                      // generic CUDA-core kernel handles it
    FactArgs fargs;
    const bool fact = smp.factored;
    if (fact) {
        pwa_status s = fill_fact_args(ctx, smp, &fargs);
        if (s != PWA_OK) return s;
    } else {
        memset(&fargs, 0, sizeof(fargs));
    }
    const bool f32 = ctx->storage == PWA_F32;
    const bool pow2 = (n & (n - 1)) == 0 && n >= 4;            // rows are whole 16-byte chunks, D = 2n
    const bool aligned = ((uintptr_t)smp.amps & 15u) == 0;
    pwa_status s;
    if (fact && smp.n_ang <= 2) s = f32 ? dispatch_nd<float, FILL_FACTORED, 2>(ctx, fargs, job) : dispatch_nd<double, FILL_FACTORED, 2>(ctx, fargs, job);
    else if (fact)            s = f32 ? dispatch_nd<float, FILL_FACTORED, 4>(ctx, fargs, job) : dispatch_nd<double, FILL_FACTORED, 4>(ctx, fargs, job);
    else if (pow2 && aligned) s = f32 ? dispatch_nd<float, FILL_STAGED, 1>(ctx, fargs, job)   : dispatch_nd<double, FILL_STAGED, 1>(ctx, fargs, job);
    else                      s = f32 ? dispatch_nd<float, FILL_ELEMENT, 1>(ctx, fargs, job)  : dispatch_nd<double, FILL_ELEMENT, 1>(ctx, fargs, job);
    if (s != PWA_OK) return s;
    *handled = true;
    return PWA_OK;
}

pwa_status launch_norm_dmma(pwa_ctx *ctx, bool *handled)
{
    GramJob job{&ctx->mc, nullptr, nullptr, false};
    return run_gram(ctx, job, handled);
}

// Fumili-style approximate Hessian over the DATA sample (V already in ctx->d_V, H_dev [2n][2n] device).
pwa_status launch_fumili(pwa_ctx *ctx, double *H_dev, bool with_norm)
{
    GramJob job{&ctx->data, ctx->d_V, H_dev, with_norm};
    bool handled = false;
    pwa_status s = run_gram(ctx, job, &handled);
    if (s != PWA_OK) return s;
    if (!handled) return fail(ctx, PWA_ERR_UNSUPPORTED, "pwa_fumili_hessian needs n <= 64");
    return PWA_OK;
}

}  // namespace pwa
