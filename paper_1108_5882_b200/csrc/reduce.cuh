// reduce.cuh — step A5 ("the final sum has to be computed in double precision ...
// tree sums as usually implemented on GPUs perform much better here"): fixed-shape fp64
// tree: per-thread running sums -> warp shuffles -> per-block partial in a fixed slot ->
// the last-arriving block sums the slots in slot order.  No floating-point atomics, so a
// launch with a fixed grid is bitwise reproducible.  The finishing block also performs step
// A7 (Norm = V^H M V, nll, gradient assembly; P:41 second term).
#pragma once
#include <cuda_runtime.h>

namespace pwa {

constexpr int kMaxWaves = 256;
constexpr int kMaxComp = 2 + 2 * kMaxWaves;

struct FinishArgs {
    double *partials;      // [gridDim.x][NC]
    unsigned *ticket;
    const double *M;       // device [n][n][2]; nullptr -> data-term-only output
    double *out;           // result record (M != nullptr) or [NC] components (M == nullptr)
    int n;
    bool eq2 = false;      // false: eq. 3 extended form; true: eq. 2 normalised form with
    double n_eq2 = 0.0;    //   N_data = n_eq2 (the number of data events, or the sum of their weights)
    // result delivery without a copy: `out` may be device-mapped pinned HOST memory; after the record is
    // written (system-scope fence) done_flag[0] = seq tells the polling host thread it is complete
    unsigned long long *done_flag = nullptr;
    unsigned long long seq = 0;
    // resident grid (data_term_tma.cu): the record goes to device-mapped host memory as 2 words per double,
    // (tag << 32 | low half), (tag << 32 | high half): complete when every word carries the tag, so neither a
    // system-scope fence nor a flag is needed
    unsigned long long *tagged = nullptr;
    unsigned tag = 0;
    const double *mv_ready = nullptr;     // (M V) already formed by this block in its shared memory (compute_mv), or nullptr
};

__device__ __forceinline__ double shfl_xor_d(double x, int m)
{
    return __shfl_xor_sync(0xffffffffu, x, m);
}

__device__ __forceinline__ double warp_sum(double x)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) x += shfl_xor_d(x, m);
    return x;
}

// (M V)_a -> s_mv[2a], s_mv[2a + 1] (shared memory, 2n doubles).  Must be called by every thread of the block; the caller
// synchronises the block before s_mv is read.  `slices` adjacent lanes share a row (coalesced reads of M, all loads
// independent), partial dot products are combined with a fixed xor tree: the result depends on (n, blockDim) only, so a
// kernel may form it early (while its first tiles are in flight) and hand it to assemble_from_totals as mv_ready.
__device__ inline void compute_mv(const double *M, const double *sV, int n, double *s_mv)
{
    const int tid = threadIdx.x, nthreads = blockDim.x;
    int slices = 1;
    while (slices * 2 <= 32 && slices * 2 * n <= nthreads && slices * 2 <= n) slices *= 2;
    const int rows_per_pass = nthreads / slices;
    const int sl = tid % slices, ra = tid / slices;
    for (int a0 = 0; a0 < n; a0 += rows_per_pass) {          // uniform trip count
        const int a = a0 + ra;
        double mr = 0.0, mi = 0.0;
        if (a < n) {
            const double2 *row = reinterpret_cast<const double2 *>(M) + (size_t)a * n;
#pragma unroll 4
            for (int b = sl; b < n; b += slices) {
                const double2 m = __ldg(row + b);
                const double vr = sV[2 * b], vi = sV[2 * b + 1];
                mr = fma(m.x, vr, mr); mr = fma(-m.y, vi, mr);
                mi = fma(m.x, vi, mi); mi = fma(m.y, vr, mi);
            }
        }
        for (int m = 1; m < slices; m <<= 1) { mr += shfl_xor_d(mr, m); mi += shfl_xor_d(mi, m); }
        if (a < n && sl == 0) { s_mv[2 * a] = mr; s_mv[2 * a + 1] = mi; }
    }
}

// Step A7 from block totals s_tot[0..2+2n) = {L_data, n_nonfinite, Re T_0, Im T_0, ...} and V in
// shared memory: M == nullptr -> copy the data-term components to out[0..2+2n); otherwise write
// the result record {nll, L_data, Norm, n_nonfinite, grad[2n]} (P:41 second term).
// Must be called by every thread of the block; s_tot and sV valid for all threads on entry.
// eq2 false: nll = -(L_data - Norm), grad = -2 conj(T) + 2 M V                      (eq. 3)
// eq2 true, n_eq2 = N_data (or sum of weights): nll = -L_data + N_data ln Norm, grad = -2 conj(T) + (2 N_data / Norm) M V   (eq. 2)
__device__ inline void assemble_from_totals(const double *s_tot, const double *sV, const double *M,
                                            double *out, int n, bool eq2 = false, double n_eq2 = 0.0,
                                            unsigned long long *done_flag = nullptr, unsigned long long seq = 0,
                                            unsigned long long *tagged = nullptr, unsigned tag = 0,
                                            const double *mv_ready = nullptr)
{
    auto put = [&](int idx, double v) {
        if (tagged != nullptr) {
            const unsigned long long t = (unsigned long long)tag << 32;
            volatile unsigned long long *p = tagged + 2 * idx;
            p[0] = t | (unsigned)__double2loint(v);
            p[1] = t | (unsigned)__double2hiint(v);
        } else out[idx] = v;
    };
    const int NC = 2 + 2 * n;
    const int tid = threadIdx.x, nthreads = blockDim.x;
    const int lane = tid & 31, warp = tid >> 5;
    __shared__ double s_mv_own[2 * kMaxWaves];
    if (M == nullptr) {
        for (int c = tid; c < NC; c += nthreads) out[c] = s_tot[c];
        if (done_flag != nullptr) {                 // record in mapped host memory: visible to the host before the flag
            __threadfence_system();
            __syncthreads();
            if (tid == 0) *reinterpret_cast<volatile unsigned long long *>(done_flag) = seq;
        }
        return;
    }
    if (mv_ready == nullptr) compute_mv(M, sV, n, s_mv_own);
    const double *s_mv = mv_ready != nullptr ? mv_ready : s_mv_own;
    __syncthreads();
    if (warp == 0) {
        double acc = 0.0;   // Norm = sum_a Re( conj(V_a) (M V)_a )
        for (int a = lane; a < n; a += 32) acc += sV[2 * a] * s_mv[2 * a] + sV[2 * a + 1] * s_mv[2 * a + 1];
        acc = warp_sum(acc);   // xor tree: every lane holds the same Norm
        const double gw = eq2 ? 2.0 * (n_eq2 / acc) : 2.0;
        // grad_a = -2 conj(T_a) + gw (M V)_a
        for (int a = lane; a < n; a += 32) {
            put(4 + 2 * a, -2.0 * s_tot[2 + 2 * a] + gw * s_mv[2 * a]);
            put(5 + 2 * a,  2.0 * s_tot[3 + 2 * a] + gw * s_mv[2 * a + 1]);
        }
        if (lane == 0) {
            put(0, eq2 ? (-s_tot[0] + n_eq2 * log(acc)) : -(s_tot[0] - acc));
            put(1, s_tot[0]);
            put(2, acc);
            put(3, s_tot[1]);
        }
        if (done_flag != nullptr && tagged == nullptr) {
            __threadfence_system();                 // every writing lane: record visible to the host before the flag
            __syncwarp();
            if (lane == 0) *reinterpret_cast<volatile unsigned long long *>(done_flag) = seq;
        }
    }
}

// s_tot[0..NC): this block's totals (valid for all threads after a __syncthreads by the
// caller).  s_red: shared scratch of at least blockDim.x doubles.  sV: V in shared
// memory [2n].  Must be called by every thread of the block.  Per-block partials live in fixed
// slots [slot][NC]; the last-arriving block (ticket) adds them in a fixed order (strided slot
// subsets per thread group, then the groups in group order).  No floating-point atomics: bitwise reproducible for a fixed launch shape.
__device__ inline void block_finish(double *s_tot, double *s_red, const double *sV, const FinishArgs &fa)
{
    const int n = fa.n, NC = 2 + 2 * n;
    const int tid = threadIdx.x, nthreads = blockDim.x;
    const int lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
    __shared__ bool s_last;

    // Programmatic dependent launch (data_term_tma.cu): this grid may have started while the previous kernel of
    // the stream was still finishing; the partial slots, the ticket and the result record are shared with it, so
    // wait for its completion (and memory flush) here.  Returns at once for a normally serialised launch.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    for (int c = tid; c < NC; c += nthreads) fa.partials[(size_t)blockIdx.x * NC + c] = s_tot[c];
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(fa.ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    // every block has arrived: re-arm the ticket for the next evaluation here, ahead of the fence below and long BEFORE the
    // record is published (in a resident grid the host may send the next command as soon as it sees the record, and the
    // first blocks of that evaluation must find the ticket at zero)
    if (tid == 0) *fa.ticket = 0u;
    __threadfence();

    // `ngroups` groups of NC adjacent threads: group g adds slots g, g + ngroups, ... of its
    // component (coalesced across the group); loads are issued in independent batches of FB
    const int nslots = (int)gridDim.x;
    constexpr int FB = 24;
    const int ngroups = nthreads / NC;
    if (ngroups >= 1) {
        const int g = tid / NC, c = tid - g * NC;
        if (g < ngroups) {
            const double *p = fa.partials + c;
            double acc = 0.0;
            for (int base = g; base < nslots; base += FB * ngroups) {
                double x[FB];
#pragma unroll
                for (int k = 0; k < FB; ++k) { const int sl = base + k * ngroups; x[k] = (sl < nslots) ? __ldcg(p + (size_t)sl * NC) : 0.0; }
#pragma unroll
                for (int k = 0; k < FB; ++k) acc += x[k];
            }
            s_red[tid] = acc;                     // == s_red[g * NC + c]
        }
        __syncthreads();
        for (int c2 = tid; c2 < NC; c2 += nthreads) {
            double t = 0.0;
            for (int g2 = 0; g2 < ngroups; ++g2) t += s_red[g2 * NC + c2];
            s_tot[c2] = t;
        }
    } else {                                      // more components than threads (generic kernel, n > 63)
        for (int c = tid; c < NC; c += nthreads) {
            const double *p = fa.partials + c;
            double acc = 0.0;
            for (int base = 0; base < nslots; base += FB) {
                double x[FB];
#pragma unroll
                for (int k = 0; k < FB; ++k) { const int sl = base + k; x[k] = (sl < nslots) ? __ldcg(p + (size_t)sl * NC) : 0.0; }
#pragma unroll
                for (int k = 0; k < FB; ++k) acc += x[k];
            }
            s_tot[c] = acc;
        }
    }
    __syncthreads();

    assemble_from_totals(s_tot, sV, fa.M, fa.out, n, fa.eq2, fa.n_eq2, fa.done_flag, fa.seq, fa.tagged, fa.tag, fa.mv_ready);
}

constexpr int kFastWaves = 64;   // == kMaxFastWaves (pwa_internal.h)

// Shared tail of every grouped data-pass kernel: per-thread (L, bad, T of the lane's waves)
// -> warp shuffles -> block totals -> block_finish.  Lanes with equal (lane % G) own the same
// waves; wave_of(idx) maps accumulator idx -> wave (or -1: not a wave, skipped).
template <int G, int W, int THREADS, typename WaveOf>
__device__ __forceinline__ void reduce_and_finish(double L, double bad, double (&tr)[W], double (&ti)[W],
                                                    WaveOf wave_of, const double *sV, const FinishArgs &fa)
{
    constexpr int NWARPS = THREADS / 32;
    __shared__ double s_warp[NWARPS][2 + 2 * kFastWaves];
    __shared__ double s_tot[2 + 2 * kFastWaves];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int NC = 2 + 2 * fa.n;
    L = warp_sum(L);
    bad = warp_sum(bad);
#pragma unroll
    for (int w = 0; w < W; ++w) {
#pragma unroll
        for (int m = G; m < 32; m <<= 1) {
            tr[w] += shfl_xor_d(tr[w], m);
            ti[w] += shfl_xor_d(ti[w], m);
        }
    }
    if (lane == 0) { s_warp[warp][0] = L; s_warp[warp][1] = bad; }
    if (lane < G) {
#pragma unroll
        for (int w = 0; w < W; ++w) {
            const int a = wave_of(w);
            if (a >= 0) { s_warp[warp][2 + 2 * a] = tr[w]; s_warp[warp][3 + 2 * a] = ti[w]; }
        }
    }
    __syncthreads();
    for (int c = threadIdx.x; c < NC; c += THREADS) {
        double acc = 0.0;
#pragma unroll
        for (int w = 0; w < NWARPS; ++w) acc += s_warp[w][c];
        s_tot[c] = acc;
    }
    __syncthreads();
    block_finish(s_tot, &s_warp[0][0], sV, fa);
}

}  // namespace pwa
