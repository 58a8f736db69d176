// data_term_tma.cu — steps A2-A5, TMA-tiled two-phase kernel.  Used for
// rows that are a whole number of 128-byte lines (fp32: n = 16, 32, 64; fp64: n = 8 ... 64).
//
//   S_i = sum_a V_a A_ia, I_i = |S_i|^2                eq. 1
//   L_data = sum_i ln I_i                              eq. 3 first term
//   T_a = sum_i A_ia / S_i                             gradient of L_data
//
// Warps work in groups of GW; a group owns a ring of NS shared-memory stages and its tiles are
// taken round-robin (tile t of the group: warp t % GW, stage t % NS), so GW tiles are being
// processed while NS-GW are in flight.  A stage is a tile of TR = 32/LPR
// consecutive events, fetched by the TMA unit (cp.async.bulk.tensor.2d, SASS UTMALDG) as CB column
// boxes of [TR rows x 128 bytes] with the 128-byte swizzle: the 16-byte chunk c of row r lands at
// slot c ^ (r & 7) of its 128-byte line.  That makes BOTH access patterns conflict-free:
//   phase 1 (lane = event, LPR lanes per row): every lane walks its own row; the 8 lanes of a
//            quarter-warp sit on 8 consecutive rows and hit 8 different slots.  S_i is formed with
//            no cross-lane traffic (LPR = 1) or one shuffle-add (LPR > 1); V comes from the constant
//            bank (kernel parameter, LPR = 1) or shared memory (LPR > 1).  ONE log and ONE
//            reciprocal per event (no redundancy); r_i = 1/S_i goes to a 16-byte smem slot.
//   phase 2 (lane = 16-byte chunk of the row = 1 or 2 waves): the warp walks the tile's rows, each
//            lane accumulates A_ia * r_i for its own waves (r_i is a broadcast load).
// The tile is read from HBM once and from shared memory twice.  Out-of-range rows of the last
// tile are zero-filled by the TMA unit and masked (r_i = 0, not counted).  Lane 0 re-arms a stage
// (with the group's tile t + NS) right after its warp has finished phase 2 of tile t and bumps the
// stage's issue counter; the next owner of the stage waits for that counter and then for the TMA
// completion barrier (no block barrier inside the loop).
// ln I_i is accumulated as a running product of mantissas plus an integer exponent sum, with one
// log per 256 events per lane (P:47 leaves the summation algorithm open; the error of the product,
// <= 256 * 2^-53 relative, is of the same order as the rounding of 256 separate logs); 1/I_i is a
// MUFU seed plus two Newton steps.  Abnormal intensities (0, denormal, inf, nan: reading C14)
// take the plain IEEE log / division path.  Reduction: reduce.cuh (A5, A7).
#include <cuda.h>
#include <cudaTypedefs.h>

#include "pwa_internal.h"
#include "reduce.cuh"
#include "stream_common.cuh"
#include "tcgen05_common.cuh"

namespace pwa {

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *tmap, int x, int y, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(tmap), "r"(x), "r"(y), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_2d_hint(uint32_t dst, const CUtensorMap *tmap, int x, int y, uint32_t bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
                 ::"r"(dst), "l"(tmap), "r"(x), "r"(y), "r"(bar), "l"(policy) : "memory");
}
// L2 residency across evaluations: the sample is re-read by every evaluation of a fit, but a sample larger than L2
// streamed through an LRU cache never hits.  With resident_rows >= 0 the first `resident_rows` rows are loaded with
// evict_last, the rest with evict_first, so that a fixed head of the sample stays in L2 from one evaluation to the
// next; resident_rows < 0: plain loads.  Measured (n = 32, fp32): 256 MB sample 51.4 -> 48.3 us with a 48 MB head,
// 102 MB sample 27.1 -> 25.3 us, 1 GB 165.8 -> 162.7 us; at 2.56 GB (cfg 4) 48 MB are 2 % of the pass and the hints
// change nothing (407 us either way, alternating A/B), so large samples load plainly.
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}

__device__ __forceinline__ double2 lds_d2(uint32_t addr)
{
    double2 r;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "r"(addr));
    return r;
}
__device__ __forceinline__ void sts_d2(uint32_t addr, double x, double y)
{
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(x), "d"(y) : "memory");
}

template <typename ST, int CB, int LPR, int THREADS, int GW, int NS>
struct TmaCfg {
    static constexpr int WPC = Chunk<ST>::WPC;
    static constexpr int CPR = CB * 8;                  // 16-byte chunks per row
    static constexpr int NW = CPR * WPC;                // waves
    static constexpr int TR = 32 / LPR;                 // rows per warp tile
    static constexpr int BOXB = TR * 128;               // bytes per column box
    static constexpr int STAGE = CB * BOXB;             // bytes per stage
    static constexpr int CPL1 = CPR / LPR;              // chunks per lane, phase 1
    static constexpr int CK2 = CPR > 32 ? CPR / 32 : 1; // chunks per lane, phase 2
    static constexpr int G2 = CPR / CK2;                // lanes per row, phase 2
    static constexpr int RPI = 32 / G2;                 // rows per phase-2 iteration
    static constexpr int NWARPS = THREADS / 32;
    static constexpr int NGRP = NWARPS / GW;              // warp groups per CTA
    static constexpr size_t SMEM = (size_t)NGRP * NS * STAGE + 1024;
    static_assert(NWARPS % GW == 0 && NS > GW - 1 && NS >= 2, "ring shape");
    static_assert(CPL1 % 8 == 0 || LPR == 1, "a lane's phase-1 share must be whole column boxes");
    static_assert(TR % 8 == 0, "swizzle atom is 8 rows");
};

// Fast 1/x for normal positive x well inside the exponent range: MUFU.RCP64H seed (~2^-20)
// + two Newton steps (error <= ~1 ulp).
__device__ __forceinline__ double fast_rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

// Resident mode (RES; for small samples the per-iteration cost is latency, not bandwidth): the grid stays on the GPU
// between evaluations and is driven through a mailbox instead of launches.  cmd_host: device-mapped pinned HOST memory,
// 4n words of (tag << 32 | 32 bits of V), tag = low half of the evaluation's sequence number; cmd_dev: the same words in
// device memory.  Warp 0 of block 0 polls cmd_host over PCIe (one round trip per poll: the command is complete when all
// words carry the new tag) and forwards the words to cmd_dev, which warp 0 of every other block polls in L2 the same way.
// The record goes back the same way (FinishArgs::tagged: tag << 32 | half a double per word, no fence and no flag: the
// host has the record when every word carries the tag).  An evaluation is exactly the body of the launched kernel (same
// grid, same tiles per CTA, same reduction tree: bitwise the same result).  The host sends the next command only after it
// has seen the record, so the evaluations of a grid never overlap.  Tag 0xffffffff in every word, or ~2 s without a
// command, ends the grid.
struct ResidentArgs {
    const unsigned long long *cmd_host;      // mapped host mailbox (read with system-scope volatile loads)
    unsigned long long *cmd_dev;             // device copy of the mailbox (forwarded by block 0)
    unsigned long long start_seq;            // sequence number at launch (commands have larger numbers)
};
// tag 0xffffffff in the mailbox = quit (the host never uses it for a command)
constexpr unsigned long long kQuit = ~0ull;
__device__ __forceinline__ unsigned long long ld_sys_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// WT: per-event weights (NEXT-3): L = sum_i w_i ln I_i, T_a = sum_i w_i A_ia / S_i.  The mantissa-product logarithm does
// not commute with weights, so a weighted event takes its own IEEE log (one per lane and tile: ~10 % more instructions).
template <typename ST, int CB, int LPR, int THREADS, int MINB, int GW, int NS, bool WT, bool RES>
__global__ void __launch_bounds__(THREADS, MINB)
k_data_term_tma(const __grid_constant__ CUtensorMap tmap, long long N, long long resident_rows,
                const __grid_constant__ VArg varg, FinishArgs fa_in, const double *__restrict__ wt, ResidentArgs res)
{
    using C = TmaCfg<ST, CB, LPR, THREADS, GW, NS>;
    constexpr int WPC = C::WPC, NW = C::NW, TR = C::TR, BOXB = C::BOXB, STAGE = C::STAGE;
    constexpr int CPL1 = C::CPL1, CK2 = C::CK2, G2 = C::G2, RPI = C::RPI, NWARPS = C::NWARPS, NGRP = C::NGRP;
    constexpr int W2 = CK2 * WPC;
    constexpr int BOX_ELEMS = 128 / (int)sizeof(ST);
    constexpr int NIT2 = TR / RPI;                     // phase-2 iterations per tile
    constexpr int U2 = (NIT2 % 2 == 0) ? 2 : 1;        // independent accumulator sets in phase 2
    constexpr int FLUSH = 256;                         // tiles between two logs of the mantissa product

    extern __shared__ unsigned char tma_smem_raw[];
    __shared__ __align__(8) unsigned long long bars[NGRP][NS];
    __shared__ volatile unsigned issued[NGRP][NS];     // number of tiles issued into each stage so far (GW > 1)
    __shared__ __align__(16) double rbuf[NWARPS][32][2];
    __shared__ __align__(16) double sV[2 * NW];
    __shared__ __align__(16) double s_mv_early[2 * NW];
    __shared__ unsigned long long s_seq;
    FinishArgs fa = fa_in;
    if (!RES) for (int t = threadIdx.x; t < 2 * NW; t += THREADS) sV[t] = varg.v[t];

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = warp / GW, wig = warp % GW;        // group in the CTA, warp in the group
    const uint32_t ring0 = ((smem_u32(tma_smem_raw) + 1023u) & ~1023u) + (uint32_t)(grp * NS) * STAGE;
    const uint32_t bar0 = smem_u32(&bars[grp][0]);
    const uint32_t rb0 = smem_u32(&rbuf[warp][0][0]);
    const uint32_t sv0 = smem_u32(sV);
    if (threadIdx.x == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
    // Let the next kernel of the stream start as soon as SMs free up: its streaming phase only reads the (constant)
    // amplitudes and its own V; everything shared with this grid is touched after griddepcontrol.wait (block_finish).
    if (!RES) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    unsigned long long last_seq = res.start_seq;
    for (int pass = 0;; ++pass) {                                 // one pass per evaluation (a single pass unless RES)
    if (RES) {
        if (warp == 0) {
            // The mailbox is 4 NW words (tag << 32 | 32 bits of V); a command is complete when every word carries the same
            // new tag (8-byte stores and loads are single transactions, any arrival order is fine): ONE round trip per poll,
            // no flag behind a fence.  Block 0 polls the host's mailbox over PCIe and forwards the words to the device
            // copy, which the other blocks poll in L2 with the same protocol.
            constexpr int WPL = (4 * NW + 31) / 32;                      // words per lane
            const unsigned long long *src = blockIdx.x == 0 ? res.cmd_host : res.cmd_dev;
            const unsigned limit = blockIdx.x == 0 ? (1u << 20) : (1u << 26);     // block 0: ~2 s of PCIe polls without a command
            unsigned long long w[WPL];
            unsigned tag = 0;
            for (unsigned spins = 0;; ++spins) {
                bool same = true;
#pragma unroll
                for (int j = 0; j < WPL; ++j) {
                    const int k = lane + 32 * j;
                    w[j] = ld_sys_u64(src + (k < 4 * NW ? k : 0));
                }
                tag = __shfl_sync(0xffffffffu, (unsigned)(w[0] >> 32), 0);
#pragma unroll
                for (int j = 0; j < WPL; ++j) same = same && (unsigned)(w[j] >> 32) == tag;
                if (__all_sync(0xffffffffu, same) && tag != (unsigned)last_seq) break;
                if (spins > limit) {
                    tag = 0xffffffffu;
#pragma unroll
                    for (int j = 0; j < WPL; ++j) w[j] = 0xffffffff00000000ull;
                    break;
                }
                if (blockIdx.x != 0) __nanosleep(40);
            }
            if (blockIdx.x == 0) {
#pragma unroll
                for (int j = 0; j < WPL; ++j) {
                    const int k = lane + 32 * j;
                    if (k < 4 * NW) *reinterpret_cast<volatile unsigned long long *>(res.cmd_dev + k) = w[j];
                }
            }
            unsigned *sV32 = reinterpret_cast<unsigned *>(sV);
#pragma unroll
            for (int j = 0; j < WPL; ++j) { const int k = lane + 32 * j; if (k < 4 * NW) sV32[k] = (unsigned)w[j]; }
            if (lane == 0) s_seq = tag == 0xffffffffu ? kQuit : last_seq + (unsigned long long)(unsigned)(tag - (unsigned)last_seq);
        }
        __syncthreads();
        const unsigned long long seq = s_seq;
        if (seq == kQuit) return;
        last_seq = seq;
        fa.seq = seq;
        fa.tag = (unsigned)seq;
    }
    if (pass == 0 && wig == 0 && lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(bar0 + 8 * s, 1); issued[grp][s] = 0; }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // tile t of this group is global tile g0 + t * gstride; warp t % GW takes it in stage t % NS
    const long long ntiles = (N + TR - 1) / TR;
    const long long gstride = (long long)gridDim.x * NGRP;
    const long long g0 = (long long)blockIdx.x * NGRP + grp;
    const long long nt_grp = (ntiles > g0) ? (ntiles - g0 + gstride - 1) / gstride : 0;   // tiles of this group
    // a resident grid keeps its mbarriers and issue counters alive across evaluations: stage s has seen
    // pass * ceil((nt_grp - s) / NS) tiles (completed barrier phases) before this pass
    auto phase0 = [&](int slot) -> unsigned {
        return RES ? (unsigned)pass * (unsigned)(nt_grp > slot ? (nt_grp - slot + NS - 1) / NS : 0) : 0u;
    };
    const uint64_t pol_keep = l2_policy_evict_last(), pol_stream = l2_policy_evict_first();
    auto issue = [&](long long t) {                              // lane 0 of the warp that owns tile t (or t - NS)
        const int slot = (int)(t % NS);
        mbar_expect_tx(bar0 + 8 * slot, STAGE);                  // OOB rows are zero-filled and still counted
        const int y = (int)((g0 + t * gstride) * TR);
        if (resident_rows < 0) {
#pragma unroll
            for (int cb = 0; cb < CB; ++cb)
                tma_load_2d(ring0 + (uint32_t)slot * STAGE + cb * BOXB, &tmap, cb * BOX_ELEMS, y, bar0 + 8 * slot);
        } else {
            const uint64_t pol = (long long)y < resident_rows ? pol_keep : pol_stream;
#pragma unroll
            for (int cb = 0; cb < CB; ++cb)
                tma_load_2d_hint(ring0 + (uint32_t)slot * STAGE + cb * BOXB, &tmap, cb * BOX_ELEMS, y, bar0 + 8 * slot, pol);
        }
        if (GW > 1) { __threadfence_block(); issued[grp][slot] = phase0(slot) + (unsigned)(t / NS) + 1u; }
    };
    if (lane == 0) {
        for (long long t = wig; t < NS && t < nt_grp; t += GW) issue(t);
    }
    // (M V) of step A7 while the first tiles are in flight: every block forms it (n^2 complex multiply-adds from the
    // L2-resident M), the block that finishes last uses its copy, and the finish loses a dependent L2 round trip
    if (fa.M != nullptr) { compute_mv(fa.M, sV, NW, s_mv_early); fa.mv_ready = s_mv_early; }

    // phase-1 coordinates: lane -> (row, part)
    const int row1 = lane % TR, part = lane / TR;
    uint32_t a1[8];                                               // per-slot address offsets of this lane's row
#pragma unroll
    for (int c = 0; c < 8; ++c)
        a1[c] = (uint32_t)row1 * 128u + (uint32_t)((c ^ (row1 & 7)) << 4) + (LPR > 1 ? (uint32_t)(part * (CPL1 / 8)) * BOXB : 0u);
    // phase-2 coordinates: lane -> (chunk(s), row selector)
    const int g2 = lane % G2, rsel = lane / G2;
    uint32_t a2[CK2]; int c2[CK2];
#pragma unroll
    for (int k = 0; k < CK2; ++k) {
        const int ch = g2 + G2 * k;
        a2[k] = (uint32_t)(ch >> 3) * BOXB;
        c2[k] = (ch & 7) << 4;
    }

    double tr[U2][W2], ti[U2][W2];
#pragma unroll
    for (int u = 0; u < U2; ++u)
#pragma unroll
        for (int w = 0; w < W2; ++w) { tr[u][w] = 0.0; ti[u][w] = 0.0; }
    double L = 0.0, bad = 0.0, P = 1.0;                          // P: running product of mantissas in [1, 2)
    int esum = 0, since = 0;                                     // sum of unbiased exponents; tiles since the last flush

    for (long long t = wig; t < nt_grp; t += GW) {
        const int slot = (int)(t % NS);
        const uint32_t parity = (uint32_t)((phase0(slot) + (unsigned)(t / NS)) & 1u);
        const uint32_t tile = ring0 + (uint32_t)slot * STAGE;
        const long long row0 = (g0 + t * gstride) * TR;
        double wv = 1.0;                                          // requested before the wait on the tile: its latency hides there
        if (WT) wv = (row0 + row1) < N ? __ldg(wt + row0 + row1) : 0.0;
        // A stage is re-armed by the warp that consumed its previous tile, which may be another warp
        // of the group: a parity wait is only unambiguous once that re-arm has happened (before it the
        // barrier can still be one phase behind, and the flipped parity would read as "complete").
        if (GW > 1) { const unsigned need = phase0(slot) + (unsigned)(t / NS) + 1u; while ((int)(issued[grp][slot] - need) < 0) { } }
        mbar_wait(bar0 + 8 * slot, parity);

        // ---------------- phase 1: S_i, ln I_i, r_i
        double sre[4] = {0.0, 0.0, 0.0, 0.0}, sim[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int i = 0; i < CPL1; ++i) {
            const uint4 q = lds128(tile + a1[i & 7] + (uint32_t)(i >> 3) * BOXB);
            double ar[WPC], ai[WPC];
            Chunk<ST>::unpack(q, ar, ai);
#pragma unroll
            for (int w = 0; w < WPC; ++w) {
                double vr, vi;
                if (LPR == 1 && !RES) { vr = varg.v[2 * (i * WPC + w)]; vi = varg.v[2 * (i * WPC + w) + 1]; }
                else { const double2 v = lds_d2(sv0 + (uint32_t)((part * CPL1 + i) * WPC + w) * 16u); vr = v.x; vi = v.y; }
                const int c = (i * WPC + w) & 1;                  // 2 x 2 independent chains per component
                sre[c] = fma(vr, ar[w], sre[c]); sre[2 + c] = fma(-vi, ai[w], sre[2 + c]);
                sim[c] = fma(vr, ai[w], sim[c]); sim[2 + c] = fma(vi, ar[w], sim[2 + c]);
            }
        }
        double sr = (sre[0] + sre[1]) + (sre[2] + sre[3]), si = (sim[0] + sim[1]) + (sim[2] + sim[3]);
#pragma unroll
        for (int m = TR; m < 32; m <<= 1) { sr += shfl_xor_d(sr, m); si += shfl_xor_d(si, m); }
        {
            const bool valid = (row0 + row1) < N;
            const bool counted = valid && part == 0;
            const double I = sr * sr + si * si;
            const int hi = __double2hiint(I);
            const unsigned ex = ((unsigned)hi >> 20) & 0x7ffu;   // I >= 0 or nan: biased exponent (sign ignored)
            const bool normal = (ex - 1u) < 0x7feu && hi > 0;    // not 0 / denormal / inf / nan / negative
            double rr, rim;
            if (WT) {                                             // weighted: plain IEEE log per event (reading C14 included)
                const double l = log(I);
                const double inv = 1.0 / I;
                rr = sr * inv * wv; rim = -si * inv * wv;
                if (counted) { L += wv * l; if (!(I > 0.0) || !isfinite(l)) bad += 1.0; }
            } else if (__all_sync(0xffffffffu, normal || !valid)) {
                const double inv = fast_rcp(valid ? I : 1.0);
                rr = sr * inv; rim = -si * inv;                   // r = conj(S) / I
                if (counted) {
                    P *= __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(I));
                    esum += (int)ex - 1023;
                }
            } else {                                              // reading C14: plain IEEE values
                const double l = log(I);
                const double inv = 1.0 / I;
                rr = sr * inv; rim = -si * inv;
                if (counted) { L += l; if (!(I > 0.0) || !isfinite(l)) bad += 1.0; }
            }
            if (!valid) { rr = 0.0; rim = 0.0; }
            if (part == 0) sts_d2(rb0 + (uint32_t)row1 * 16u, rr, rim);
            if (++since == FLUSH) { L += log(P); P = 1.0; since = 0; }
        }
        __syncwarp();

        // ---------------- phase 2: T_a += A_ia r_i
#pragma unroll 2
        for (int it = 0; it < NIT2; it += U2) {
#pragma unroll
            for (int u = 0; u < U2; ++u) {
                const int r = (it + u) * RPI + rsel;
                const double2 rv = lds_d2(rb0 + (uint32_t)r * 16u);
                const uint32_t rowa = tile + (uint32_t)r * 128u;
                const int xr = (r & 7) << 4;
#pragma unroll
                for (int k = 0; k < CK2; ++k) {
                    const uint4 q = lds128(rowa + a2[k] + (uint32_t)(c2[k] ^ xr));
                    double ar[WPC], ai[WPC];
                    Chunk<ST>::unpack(q, ar, ai);
#pragma unroll
                    for (int w = 0; w < WPC; ++w) {
                        tr[u][k * WPC + w] = fma(ar[w], rv.x, tr[u][k * WPC + w]); tr[u][k * WPC + w] = fma(-ai[w], rv.y, tr[u][k * WPC + w]);
                        ti[u][k * WPC + w] = fma(ar[w], rv.y, ti[u][k * WPC + w]); ti[u][k * WPC + w] = fma(ai[w], rv.x, ti[u][k * WPC + w]);
                    }
                }
            }
        }
        __syncwarp();                                             // tile and rbuf fully consumed
        if (lane == 0 && t + NS < nt_grp) issue(t + NS);
    }
    L += log(P) + 0.6931471805599453094 * (double)esum;
    double trs[W2], tis[W2];
#pragma unroll
    for (int w = 0; w < W2; ++w) { trs[w] = tr[0][w]; tis[w] = ti[0][w]; if (U2 > 1) { trs[w] += tr[U2 - 1][w]; tis[w] += ti[U2 - 1][w]; } }
    auto wave_of = [&](int idx) { return (g2 + G2 * (idx / WPC)) * WPC + (idx % WPC); };
    reduce_and_finish<G2, W2, THREADS>(L, bad, trs, tis, wave_of, sV, fa);
    if (!RES) return;
    __syncthreads();                                              // every warp is past its last barrier wait: the ring can be re-armed
    }
}

// ---- host side: tensor map ------------------------------------------------------------------------
static pwa_status make_tmap(pwa_ctx *ctx, CUtensorMap *out, const void *base, bool f32, int n, long long N, int box_rows)
{
    PFN_cuTensorMapEncodeTiled_v12000 enc = tc::tensor_map_encoder();
    if (!enc) return fail(ctx, PWA_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
    const cuuint64_t gdim[2] = {(cuuint64_t)(2 * n), (cuuint64_t)N};
    const cuuint64_t gstride[1] = {(cuuint64_t)(2 * n) * (f32 ? 4u : 8u)};
    const cuuint32_t box[2] = {(cuuint32_t)(f32 ? 32 : 16), (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(out, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(base),
                     gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                     CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, PWA_ERR_CUDA, "cuTensorMapEncodeTiled failed (code " + std::to_string((int)r) + ")");
    return PWA_OK;
}

template <typename ST, int CB, int LPR, int THREADS, int MINB, int GW, int NS>
static pwa_status launch_tma(pwa_ctx *ctx, const VArg &varg, const FinishArgs &fa_in, bool resident)
{
    using C = TmaCfg<ST, CB, LPR, THREADS, GW, NS>;
    const bool weighted = ctx->data.weights != nullptr;
    if (resident && weighted) return fail(ctx, PWA_ERR_UNSUPPORTED, "resident evaluation does not take event weights");
    auto kern = resident ? k_data_term_tma<ST, CB, LPR, THREADS, MINB, GW, NS, false, true>
              : weighted ? k_data_term_tma<ST, CB, LPR, THREADS, MINB, GW, NS, true, false>
                         : k_data_term_tma<ST, CB, LPR, THREADS, MINB, GW, NS, false, false>;
    const long long N = ctx->data.n_events;
    // per-instantiation, per-device launch plan: attribute + occupancy are queried once
    static int s_occ2[3][64] = {{0}};
    int &occ = s_occ2[resident ? 2 : weighted ? 1 : 0][ctx->device & 63];
    if (occ == 0) {
        PWA_CUDA(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM));
        int o = 0;
        PWA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kern, THREADS, C::SMEM));
        occ = o < 1 ? 1 : o;
    }
    static_assert(sizeof(CUtensorMap) <= sizeof(ctx->tmap_cache.map), "tensor map cache too small");
    auto &tc = ctx->tmap_cache;
    if (!tc.valid || tc.base != ctx->data.amps || tc.n_events != N || tc.box_rows != C::TR) {
        pwa_status s = make_tmap(ctx, reinterpret_cast<CUtensorMap *>(tc.map), ctx->data.amps, sizeof(ST) == 4, ctx->n, N, C::TR);
        if (s != PWA_OK) return s;
        tc.base = ctx->data.amps; tc.n_events = N; tc.box_rows = C::TR; tc.valid = true;
    }
    const long long ntiles = (N + C::TR - 1) / C::TR;
    long long want = (ntiles + C::NGRP - 1) / C::NGRP;
    long long grid = (long long)ctx->sm_count * occ;
    if (want < grid) grid = want;
    if (grid < 1) grid = 1;
    FinishArgs fa = fa_in;
    pwa_status s = ensure_partials(ctx, (size_t)n_components(ctx->n) * (size_t)grid);
    if (s != PWA_OK) return s;
    fa.partials = ctx->d_partials;
    // programmatic stream serialisation: the grid may begin while its predecessor drains (see the kernel's prologue)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(THREADS); cfg.dynamicSmemBytes = C::SMEM; cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    // measured: up to ~1 GB per pass the overlap wins (51.4 vs 56.0 us at 256 MB, 162 vs 166 us at 1 GB); beyond, the early
    // successor CTAs disturb the tail of the running grid (0.417 vs 0.406 ms at 2.56 GB), so large samples launch plainly.
    // "data_term" = 98: experiment switch, always plain serialisation.
    const bool pdl = !resident && ctx->opt_data_term != 98 && (size_t)N * (size_t)ctx->n * 2 * sizeof(ST) <= ((size_t)1 << 30);
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr; cfg.numAttrs = 1;
    // head of the sample kept in L2 between evaluations (see l2_policy_evict_last): 48 MB by default for samples that do
    // not fit L2 anyway but are small enough for the hints to pay (<= 1 GiB); "l2_resident_mb" overrides (0 = plain loads)
    const size_t sample_bytes = (size_t)N * (size_t)ctx->n * 2 * sizeof(ST);
    const long long row_bytes = (long long)ctx->n * 2 * (long long)sizeof(ST);
    long long resident_rows = -1;
    if (ctx->opt_l2_resident_mb > 0) resident_rows = ((long long)ctx->opt_l2_resident_mb << 20) / row_bytes;
    else if (ctx->opt_l2_resident_mb < 0 && sample_bytes <= ((size_t)1 << 30) && sample_bytes > ((size_t)64 << 20)) resident_rows = ((long long)48 << 20) / row_bytes;
    ResidentArgs res{nullptr, nullptr, 0ull};
    if (resident) { res.cmd_host = ctx->dev_cmd_host; res.cmd_dev = ctx->d_cmd; res.start_seq = ctx->seq; }
    PWA_CUDA(ctx, cudaLaunchKernelEx(&cfg, kern, *reinterpret_cast<const CUtensorMap *>(tc.map), N, resident_rows, varg, fa,
                                     (const double *)ctx->data.weights, res));
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

// One configuration per (storage, n): the fastest of the variants measured in round 1 (profiles/r1b_summary.md).
pwa_status launch_data_term_tma(pwa_ctx *ctx, const VArg &varg, const FinishArgs &fa, bool *handled, bool resident)
{
    *handled = false;
    const int n = ctx->n;
    const bool f32 = ctx->storage == PWA_F32;
    const long long N = ctx->data.n_events;
    if (N < 1 || N > 0x7fffffffLL || ((uintptr_t)ctx->data.amps & 15u) != 0) return PWA_OK;
    const int row_bytes = 2 * n * (f32 ? 4 : 8);
    if (row_bytes % 128 != 0 || row_bytes > 1024 || (n & (n - 1)) != 0) return PWA_OK;
    *handled = true;
    //                         ST    CB LPR THREADS MINB GW NS     stage bytes
    if (f32) {
        switch (n) {
        case 16: return launch_tma<float, 1, 1, 256, 2, 1, 3>(ctx, varg, fa, resident);      //  4 KB
        case 32: return launch_tma<float, 2, 1, 512, 1, 2, 3>(ctx, varg, fa, resident);      //  8 KB, 16 warps
        case 64: return launch_tma<float, 4, 2, 512, 1, 2, 3>(ctx, varg, fa, resident);      //  8 KB, 16 warps, groups of 2
        }
    } else {
        switch (n) {
        case 8:  return launch_tma<double, 1, 1, 256, 2, 1, 3>(ctx, varg, fa, resident);
        case 16: return launch_tma<double, 2, 2, 512, 1, 2, 3>(ctx, varg, fa, resident);
        case 32: return launch_tma<double, 4, 2, 512, 1, 2, 3>(ctx, varg, fa, resident);
        case 64: return launch_tma<double, 8, 4, 512, 1, 2, 3>(ctx, varg, fa, resident);
        }
    }
    *handled = false;
    return PWA_OK;
}

}  // namespace pwa
