// norm_i8.cu — step A6 on the 5th-generation tensor cores:
// the normalisation matrix
//     M_ab = (1/N_gen) sum_j conj(B_ja) B_jb              eq. 3 inner bracket (reading C1)
// of an fp32-STORED, constant-resonance MC sample (built once per fit; single-precision
// amplitudes, double-precision sums), as an error-free integer contraction:
//
//   * real embedding as in norm_dmma.cu: B viewed as real [N_acc x D], D = 2n, P = B^T B (D x D).
//     For D < 128, G = 128/D consecutive events are viewed as ONE row of 128 reals (the diagonal
//     D x D blocks of the 128 x 128 Gram are added at the end), so the kernel always sees 128 columns.
//   * every column p has a power-of-two scale 2^s_p (from max_j |B_jp|, found once at upload) and
//     q_jp = rint(B_jp 2^s_p) is a 32-bit integer, |q| <= 2^31 - 2^24: fixed point with 31 bits
//     below the column maximum.  q = d0 + 2^8 d1 + 2^16 d2 + 2^24 d3 with BALANCED digits
//     d in [-128, 127] ("Ozaki" slicing); the four int8 digit planes D0..D3 of a 64-event tile are
//     written to shared memory in the UMMA canonical MN-major / 128-byte-swizzle layout.
//   * tcgen05.mma.kind::i8 (int8 x int8 -> int32 in TMEM, exact) forms, per 32-event K step,
//         acc6 += D3^T D3                       order t = u + v = 6
//         acc5 += D3^T D2                       t = 5   (P5 = acc5 + acc5^T)
//         acc4 += 2 D3^T D1 + D2^T D2           t = 4   (P4 = (acc4 + acc4^T) / 2)
//         acc3 += D3^T D0 + D2^T D1             t = 3   (P3 = acc3 + acc3^T)
//     4 accumulators x 128 columns = all 512 TMEM columns; 7 products (M = N = 128, K = 32) per K
//     step instead of the 16 digit pairs, using the symmetry of the Gram matrix, issued as three
//     N = 256 MMAs over adjacent planes / adjacent accumulators plus one N = 128 MMA.  Orders t <= 2 are
//     dropped: |dropped| <= 3 * 2^-32 * (1 + 2^-7) c_p c_q per event, c_p = 2^(31 - s_p) in
//     (max|B_p|, 2 max|B_p|]; the quantisation adds <= 2^-32 (c_p |B_q| + c_q |B_p|).  Both are
//     far below the 1e-6 tolerance of fp32 storage (BASELINE.json north_star) for any realistic
//     max/rms ratio; pwa_norm_error_bound() evaluates the bound for the uploaded sample.
//     The dropped terms are zero-mean EXCEPT on the diagonal p = q, where sum_e d1^2 > 0 is a
//     systematic bias (measured 5e-9 of max|M|); the converters therefore also accumulate the exact
//     t = 2 diagonal, sum_e (d1^2 + 2 d0 d2), with one dp4a per element, and it is added back.
//   * int32 cannot overflow: <= 3 * 2^14 per event into acc2, flushed every FT * 64 = 32768 events
//     (3 * 2^14 * 2^15 < 2^31) to an fp64 per-CTA slot; slots are summed in slot order
//     (bitwise reproducible), symmetrised, unscaled and folded to the complex Hermitian M.
//
// Warp roles (one persistent CTA per SM): NCW converter/epilogue warps (fp32 tile -> digit planes;
// TMEM -> fp64 slot), one TMA producer warp (cp.async.bulk.tensor ring of fp32 tiles), one MMA
// issuer warp (owns the TMEM allocation; a single lane issues tcgen05.mma / tcgen05.commit).
#include <cuda.h>
#include <cudaTypedefs.h>
#include <math.h>
#include <string.h>

#include "pwa_internal.h"
#include "stream_common.cuh"
#include "tcgen05_common.cuh"

namespace pwa {

namespace i8 {

using namespace tc;

constexpr int TE = 64;                       // super-rows (K) per tile
constexpr int ROWB = 512;                    // bytes of one fp32 super-row (128 reals)
constexpr int STG_BYTES = TE * ROWB;         // 32 KB fp32 tile
constexpr int PLANE = TE * 128;              // 8 KB: one int8 digit plane of a tile
constexpr int SL_BYTES = 4 * PLANE;          // 32 KB: four digit planes (the three-plane variant leaves the fourth unused)
constexpr int NSTG = 3;                      // fp32 tile ring
constexpr int NSL = 3;                       // digit-plane ring
constexpr int FT = 512;                      // tiles between two TMEM flushes (32768 events)
constexpr int NCW = 8;                       // converter / epilogue warps
constexpr int THREADS = (NCW + 2) * 32;
constexpr size_t SMEM = 1024 + (size_t)NSTG * STG_BYTES + (size_t)NSL * SL_BYTES;

struct Scales { float s[128]; int one; };    // 2^s_p per real column of the 128-wide view; one = 1 (a runtime 1 keeps the digit-offset add on the IMAD pipe)

// One digit plane (or a 32-row K step of it) as an MN-major operand (tcgen05_common.cuh): one plane is exactly one
// 128-byte atom along MN; an N = 256 operand continues in the NEXT plane (LBO = PLANE), so [D_v | D_v+1] is one B
// operand and its two products land in adjacent accumulators.
__device__ __forceinline__ uint64_t plane_desc(uint32_t smem_addr) { return desc_mnmajor(smem_addr, PLANE); }
constexpr uint32_t kIdesc128 = idesc_i8(128, true, true), kIdesc256 = idesc_i8(256, true, true);   // both operands MN-major

// ---- the kernel -------------------------------------------------------------------------------
// tmap: fp32 [rows][128] view of the MC sample, box = [TE rows][128 floats], no swizzle.
// slots: [gridDim.x][128][128] doubles, Y = 2^23 acc0 + 2^16 acc1 + 2^7 acc2 + acc3 summed over the
// CTA's flushes (P = 2^24 (Y + Y^T) in units of 2^-(s_p + s_q)).
// dslots: [gridDim.x][NCW][128] doubles, the t = 2 diagonal per converter warp (P_pp += 2^16 * sum).
// NP = 4: the scheme above.  NP = 3 (option "norm" = 3): q = rint(B 2^(s_p - 8)) has 24 bits below the column maximum and
// three balanced digits; per K step
//     acc4 += D2^T D2  (t = 4),  acc3 += D2^T D1  (t = 3)      one N = 256 MMA, D2^T [D1 | D2]
//     acc2a += D2^T D0,  acc2b += D1^T D1           (t = 2)      two N = 128 MMAs
// = 4 products instead of 7 and 56 KB instead of 88 KB of operand reads per tile; orders t <= 1 are dropped (the exact
// t = 0 diagonal sum_e d0^2 is added back).  Y = 2^16 acc4 + 2^9 acc3 + 2 acc2a + acc2b, P = 2^31 (Y + Y^T) 2^-(s_p + s_q).
template <int NP>
__global__ void __launch_bounds__(THREADS, 1)
k_norm_i8(const __grid_constant__ CUtensorMap tmap, long long ntiles, const __grid_constant__ Scales sc,
          double *__restrict__ slots, double *__restrict__ dslots)
{
    extern __shared__ unsigned char i8_smem_raw[];
    __shared__ __align__(8) unsigned long long bars[2 * NSTG + 2 * NSL + 2];
    __shared__ uint32_t tmem_base_s;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t base = (smem_u32(i8_smem_raw) + 1023u) & ~1023u;
    const uint32_t stg0 = base, sl0 = base + NSTG * STG_BYTES;
    const uint32_t b_stg_full = smem_u32(&bars[0]), b_stg_empty = b_stg_full + 8 * NSTG;
    const uint32_t b_sl_full = b_stg_empty + 8 * NSTG, b_sl_empty = b_sl_full + 8 * NSL;
    const uint32_t b_acc_full = b_sl_empty + 8 * NSL, b_acc_empty = b_acc_full + 8;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTG; ++s) { mbar_init(b_stg_full + 8 * s, 1); mbar_init(b_stg_empty + 8 * s, NCW); }
        for (int s = 0; s < NSL; ++s) { mbar_init(b_sl_full + 8 * s, NCW); mbar_init(b_sl_empty + 8 * s, 1); }
        mbar_init(b_acc_full, 1); mbar_init(b_acc_empty, NCW);
        fence_async_smem();
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmap) : "memory");
    }
    if (warp == NCW + 1) tmem_alloc(smem_u32(&tmem_base_s), 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem0 = tmem_base_s;

    // contiguous tile range of this CTA
    const long long per = ntiles / gridDim.x, rem = ntiles % gridDim.x;
    const long long t_begin = (long long)blockIdx.x * per + (blockIdx.x < rem ? blockIdx.x : rem);
    const long long nt = per + (blockIdx.x < rem ? 1 : 0);

    if (warp == NCW) {
        // ===== TMA producer =====
        if (lane == 0) {
            for (long long t = 0; t < nt; ++t) {
                const int s = (int)(t % NSTG);
                if (t >= NSTG) mbar_wait(b_stg_empty + 8 * s, (uint32_t)((t / NSTG - 1) & 1));
                mbar_expect_tx(b_stg_full + 8 * s, STG_BYTES);
                asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                             ::"r"(stg0 + (uint32_t)s * STG_BYTES), "l"(&tmap), "r"(0), "r"((int)((t_begin + t) * TE)),
                               "r"(b_stg_full + 8 * s) : "memory");
            }
        }
    } else if (warp == NCW + 1) {
        // ===== MMA issuer =====
        if (lane == 0) {
            for (long long t = 0; t < nt; ++t) {
                const int b = (int)(t % NSL);
                const bool first = (t % FT) == 0;
                mbar_wait(b_sl_full + 8 * b, (uint32_t)((t / NSL) & 1));
                if (first && t > 0) mbar_wait(b_acc_empty, (uint32_t)((t / FT - 1) & 1));
                tc_fence_after();
                const uint32_t pl = sl0 + (uint32_t)b * SL_BYTES;
#pragma unroll
                for (int kk = 0; kk < TE / 32; ++kk) {
                    const uint32_t koff = (uint32_t)kk * 32u * 128u;
                    const uint64_t d0 = plane_desc(pl + 0 * PLANE + koff), d1 = plane_desc(pl + 1 * PLANE + koff);
                    const uint64_t d2 = plane_desc(pl + 2 * PLANE + koff), d3 = plane_desc(pl + 3 * PLANE + koff);
                    const uint32_t acc = (first && kk == 0) ? 0u : 1u;
                    if (NP == 4) {
                        // accumulators by ascending order: t = 3 at column 0, t = 4 at 128, t = 5 at 256, t = 6 at 384
                        umma_i8(tmem0 + 256, d3, d2, kIdesc256, acc);      // D3^T [D2 | D3] -> t = 5 | t = 6
                        umma_i8(tmem0 + 0,   d3, d0, kIdesc256, acc);      // D3^T [D0 | D1] -> t = 3 | t = 4
                        umma_i8(tmem0 + 128, d3, d1, kIdesc128, 1u);       // second D3^T D1  -> t = 4
                        umma_i8(tmem0 + 0,   d2, d1, kIdesc256, 1u);       // D2^T [D1 | D2] -> t = 3 | t = 4
                    } else {
                        // D2^T D0 at column 0, D1^T D1 at 128, t = 3 at 256, t = 4 at 384
                        umma_i8(tmem0 + 256, d2, d1, kIdesc256, acc);      // D2^T [D1 | D2] -> t = 3 | t = 4
                        umma_i8(tmem0 + 0,   d2, d0, kIdesc128, acc);      // D2^T D0        -> t = 2
                        umma_i8(tmem0 + 128, d1, d1, kIdesc128, acc);      // D1^T D1        -> t = 2
                    }
                }
                umma_commit(b_sl_empty + 8 * b);
                if ((t % FT) == FT - 1 || t == nt - 1) umma_commit(b_acc_full);
            }
        }
    } else {
        // ===== converters / epilogue =====
        const int one = sc.one;
        float scl[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) scl[i] = sc.s[4 * lane + i];
        double *slot = slots + (size_t)blockIdx.x * 128 * 128;
        double *dslot = dslots + ((size_t)blockIdx.x * NCW + warp) * 128 + 4 * lane;
        int dg[4] = {0, 0, 0, 0};                                      // t = 2 diagonal of this lane's 4 columns
        const uint32_t chunk_off = (uint32_t)(lane & 3) * 4u;          // byte offset inside the 16-byte chunk
        const uint32_t chunk_id = (uint32_t)(lane >> 2);               // 16-byte chunk of the 128-byte plane row
        for (long long t = 0; t < nt; ++t) {
            const int s = (int)(t % NSTG), b = (int)(t % NSL);
            mbar_wait(b_stg_full + 8 * s, (uint32_t)((t / NSTG) & 1));
            if (t >= NSL) mbar_wait(b_sl_empty + 8 * b, (uint32_t)((t / NSL - 1) & 1));
            const uint32_t src = stg0 + (uint32_t)s * STG_BYTES + (uint32_t)lane * 16u;
            const uint32_t dst = sl0 + (uint32_t)b * SL_BYTES;
            uint4 raw[TE / NCW];
#pragma unroll
            for (int r = 0; r < TE / NCW; ++r) raw[r] = lds128(src + (uint32_t)(warp + r * NCW) * ROWB);
#pragma unroll
            for (int r = 0; r < TE / NCW; ++r) {
                const uint32_t e = (uint32_t)(warp + r * NCW);
                // balanced digits: NP = 4: bytes d0 d1 d2 d3; NP = 3: bytes d0 d1 d2 (byte 3 is the sign extension of d2, unused)
                constexpr int OFS = NP == 4 ? 0x00808080 : 0x00008080;
                const uint32_t w0 = (uint32_t)(__float2int_rn(__uint_as_float(raw[r].x) * scl[0]) * one + OFS) ^ (uint32_t)OFS;
                const uint32_t w1 = (uint32_t)(__float2int_rn(__uint_as_float(raw[r].y) * scl[1]) * one + OFS) ^ (uint32_t)OFS;
                const uint32_t w2 = (uint32_t)(__float2int_rn(__uint_as_float(raw[r].z) * scl[2]) * one + OFS) ^ (uint32_t)OFS;
                const uint32_t w3 = (uint32_t)(__float2int_rn(__uint_as_float(raw[r].w) * scl[3]) * one + OFS) ^ (uint32_t)OFS;
                if (NP == 4) {
                    // exact t = 2 diagonal: d0 d2 + d1 d1 + d2 d0 per element (<= 3 * 2^14, 4096 rows per warp and flush)
                    dg[0] = __dp4a((int)w0, (int)__byte_perm(w0, 0u, 0x4012), dg[0]);
                    dg[1] = __dp4a((int)w1, (int)__byte_perm(w1, 0u, 0x4012), dg[1]);
                    dg[2] = __dp4a((int)w2, (int)__byte_perm(w2, 0u, 0x4012), dg[2]);
                    dg[3] = __dp4a((int)w3, (int)__byte_perm(w3, 0u, 0x4012), dg[3]);
                } else {
                    // exact t = 0 diagonal: d0 d0 per element (<= 2^14)
                    dg[0] = __dp4a((int)(w0 & 0xffu), (int)w0, dg[0]);
                    dg[1] = __dp4a((int)(w1 & 0xffu), (int)w1, dg[1]);
                    dg[2] = __dp4a((int)(w2 & 0xffu), (int)w2, dg[2]);
                    dg[3] = __dp4a((int)(w3 & 0xffu), (int)w3, dg[3]);
                }
                const uint32_t t0 = __byte_perm(w0, w1, 0x5140), t1 = __byte_perm(w2, w3, 0x5140);
                const uint32_t t2 = __byte_perm(w0, w1, 0x7362), t3 = __byte_perm(w2, w3, 0x7362);
                const uint32_t a = dst + e * 128u + ((chunk_id ^ (e & 7u)) << 4) + chunk_off;
                asm volatile("st.shared.u32 [%0], %1;" ::"r"(a + 0 * PLANE), "r"(__byte_perm(t0, t1, 0x5410)) : "memory");
                asm volatile("st.shared.u32 [%0], %1;" ::"r"(a + 1 * PLANE), "r"(__byte_perm(t0, t1, 0x7632)) : "memory");
                asm volatile("st.shared.u32 [%0], %1;" ::"r"(a + 2 * PLANE), "r"(__byte_perm(t2, t3, 0x5410)) : "memory");
                if (NP == 4) asm volatile("st.shared.u32 [%0], %1;" ::"r"(a + 3 * PLANE), "r"(__byte_perm(t2, t3, 0x7632)) : "memory");
            }
            fence_async_smem();                       // digit planes -> visible to the tensor core (async proxy)
            __syncwarp();
            if (lane == 0) { mbar_arrive(b_stg_empty + 8 * s); mbar_arrive(b_sl_full + 8 * b); }

            if ((t % FT) == FT - 1 || t == nt - 1) {
                // ----- flush: TMEM -> fp64 slot (this warp: lane quarter warp % 4, column half warp / 4) -----
                const long long chunk = t / FT;
#pragma unroll
                for (int i = 0; i < 4; ++i) { dslot[i] = (chunk > 0 ? dslot[i] : 0.0) + (double)dg[i]; dg[i] = 0; }
                mbar_wait(b_acc_full, (uint32_t)(chunk & 1));
                tc_fence_after();
                const int m = 32 * (warp & 3) + lane;
                constexpr int CPW = 128 / (NCW / 4);                       // columns per warp
                const int c_begin = (warp >> 2) * CPW;
                const uint32_t trow = tmem0 + ((uint32_t)(32 * (warp & 3)) << 16);
                for (int c0 = c_begin; c0 < c_begin + CPW; c0 += 16) {
                    int32_t a0[16], a1[16], a2[16], a3[16];
                    tmem_ld16(trow + 3 * 128 + c0, a0);            // a0: t = 6, a1: t = 5, a2: t = 4, a3: t = 3
                    tmem_ld16(trow + 2 * 128 + c0, a1);
                    tmem_ld16(trow + 1 * 128 + c0, a2);
                    tmem_ld16(trow + 0 * 128 + c0, a3);
                    tmem_ld_wait();
                    double *yp = slot + (size_t)m * 128 + c0;
#pragma unroll
                    for (int j = 0; j < 16; j += 2) {
                        // NP = 4: 2^23 t6 + 2^16 t5 + 2^7 t4 + t3;  NP = 3: 2^16 t4 + 2^9 t3 + (D1^T D1 + 2 D2^T D0)
                        constexpr double W0 = NP == 4 ? 8388608.0 : 65536.0, W1 = NP == 4 ? 65536.0 : 512.0, W2 = NP == 4 ? 128.0 : 1.0, W3 = NP == 4 ? 1.0 : 2.0;
                        double y0 = (double)a0[j] * W0 + (double)a1[j] * W1 + ((double)a2[j] * W2 + (double)a3[j] * W3);
                        double y1 = (double)a0[j + 1] * W0 + (double)a1[j + 1] * W1 + ((double)a2[j + 1] * W2 + (double)a3[j + 1] * W3);
                        if (chunk > 0) { const double2 old = *reinterpret_cast<const double2 *>(yp + j); y0 += old.x; y1 += old.y; }
                        *reinterpret_cast<double2 *>(yp + j) = make_double2(y0, y1);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(b_acc_empty);
            }
        }
        if (nt == 0) {                                   // a CTA without tiles still owns a slot: zero it
            double *yp = slot;
            for (int i = threadIdx.x; i < 128 * 128; i += NCW * 32) yp[i] = 0.0;
#pragma unroll
            for (int i = 0; i < 4; ++i) dslot[i] = 0.0;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == NCW + 1) { tc_fence_after(); tmem_dealloc(tmem0, 512); }
}

// ---- column maxima (once per upload) -------------------------------------------------------------
// cmax[p] = max_j |B_jp| as the bit pattern of a non-negative float (ordered like unsigned integers);
// a NaN anywhere gives 0x7fc00000 or larger and disables the path.
__global__ void __launch_bounds__(256)
k_colmax_f32(const float *__restrict__ B, long long nfloats, int D, unsigned *__restrict__ cmax)
{
    __shared__ unsigned s_max[128];
    if (threadIdx.x < 128) s_max[threadIdx.x] = 0u;
    __syncthreads();
    // thread owns the 4 columns (4 * tid) % D .. + 3 for all its float4 (grid stride is a multiple of D floats)
    const long long nvec = nfloats / 4;
    const long long stride = (long long)gridDim.x * 256;
    unsigned m0 = 0, m1 = 0, m2 = 0, m3 = 0;
    for (long long v = (long long)blockIdx.x * 256 + threadIdx.x; v < nvec; v += stride) {
        const uint4 q = ldg_stream(reinterpret_cast<const uint4 *>(B) + v);
        m0 = max(m0, q.x & 0x7fffffffu); m1 = max(m1, q.y & 0x7fffffffu);
        m2 = max(m2, q.z & 0x7fffffffu); m3 = max(m3, q.w & 0x7fffffffu);
    }
    const int c = (int)((4LL * threadIdx.x) % D);     // 256 * 4 and the grid stride are multiples of D (D | 128)
    atomicMax(&s_max[c], m0); atomicMax(&s_max[c + 1], m1); atomicMax(&s_max[c + 2], m2); atomicMax(&s_max[c + 3], m3);
    __syncthreads();
    if ((int)threadIdx.x < D) atomicMax(&cmax[threadIdx.x], s_max[threadIdx.x]);
}

// ---- final sum over slots (fixed order) -----------------------------------------------------------
// Ysum[p][q] = sum_slots Y; thread per element, 4 independent partial sums, combined in a fixed order.
// 256 threads = 32 elements x 8 slot phases: thread (el, ph) adds slots ph, ph + 8, ... with four
// independent loads in flight, the 8 phases are then added in phase order (a fixed tree: bitwise
// reproducible for a fixed grid).  Blocks 0..511: Y (16384 elements); blocks 512..515: the diagonal
// correction (128 elements, nslots * NCW partial rows).
__global__ void __launch_bounds__(256)
k_i8_slot_sum(const double *__restrict__ slots, int nslots, double *__restrict__ ysum,
              const double *__restrict__ dslots, double *__restrict__ dsum)
{
    __shared__ double s_ph[8][33];
    const int el = threadIdx.x & 31, ph = threadIdx.x >> 5;
    const double *src; size_t stride; int cnt; double *dst;
    if (blockIdx.x < 512) { const int idx = blockIdx.x * 32 + el; src = slots + idx; stride = 16384; cnt = nslots; dst = ysum + idx; }
    else { const int idx = (blockIdx.x - 512) * 32 + el; src = dslots + idx; stride = 128; cnt = nslots * NCW; dst = dsum + idx; }
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int s = ph;
    for (; s + 24 < cnt; s += 32) {
        const double x0 = __ldcg(src + (size_t)s * stride),        x1 = __ldcg(src + (size_t)(s + 8) * stride);
        const double x2 = __ldcg(src + (size_t)(s + 16) * stride), x3 = __ldcg(src + (size_t)(s + 24) * stride);
        a0 += x0; a1 += x1; a2 += x2; a3 += x3;
    }
    for (; s < cnt; s += 8) a0 += __ldcg(src + (size_t)s * stride);
    s_ph[ph][el] = (a0 + a1) + (a2 + a3);
    __syncthreads();
    if (ph == 0) {
        double t = 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) t += s_ph[q][el];
        *dst = t;
    }
}

struct Exps { int e[128]; };                   // s_p of the 128-wide view

// P[p][q] (D x D) = sum over the G diagonal blocks of 2^(24 - s_p - s_q) (Y + Y^T), plus the exact
// fp64 products of the n_tail events that do not fill a 128-real row; then the complex fold
//   Re M_ab = P[2a][2b] + P[2a+1][2b+1],  Im M_ab = P[2a][2b+1] - P[2a+1][2b]   (norm_dmma.cu, DESIGN 6.3)
// evaluated for a <= b and mirrored, so M is exactly Hermitian.
__global__ void __launch_bounds__(256)
k_i8_assemble(const double *__restrict__ ysum, const double *__restrict__ dsum, const __grid_constant__ Exps ex, int n,
              const float *__restrict__ tail, int n_tail, double inv_ngen, double *__restrict__ M, int yshift)
{
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= n * n) return;
    const int a = idx / n, b = idx % n;
    if (a > b) return;
    const int D = 2 * n, G = 128 / D;
    auto P = [&](int p, int q) {
        double acc = 0.0;
        for (int g = 0; g < G; ++g) {
            const int pp = g * D + p, qq = g * D + q;
            acc += (ysum[pp * 128 + qq] + ysum[qq * 128 + pp]) * exp2((double)(yshift - ex.e[pp] - ex.e[qq]));   // 24 (four planes) or 31 (three)
            if (p == q) acc += dsum[pp] * exp2((double)(16 - 2 * ex.e[pp]));
        }
        for (int j = 0; j < n_tail; ++j) acc += (double)tail[(size_t)j * D + p] * (double)tail[(size_t)j * D + q];
        return acc;
    };
    const double re = (P(2 * a, 2 * b) + P(2 * a + 1, 2 * b + 1)) * inv_ngen;
    const double im = (a == b) ? 0.0 : (P(2 * a, 2 * b + 1) - P(2 * a + 1, 2 * b)) * inv_ngen;
    M[((size_t)a * n + b) * 2] = re;  M[((size_t)a * n + b) * 2 + 1] = im;
    if (a != b) { M[((size_t)b * n + a) * 2] = re;  M[((size_t)b * n + a) * 2 + 1] = -im; }
}

}  // namespace i8

// ---- host side ----------------------------------------------------------------------------------
static bool i8_shape_ok(const pwa_ctx *ctx)
{
    const int D = 2 * ctx->n;
    return ctx->storage == PWA_F32 && !ctx->mc.factored && ctx->mc.weights == nullptr && (D == 32 || D == 64 || D == 128) &&
           ctx->mc.n_events > 0 && ((uintptr_t)ctx->mc.amps & 15u) == 0;
}

// Column maxima of an fp32-stored [n_events x D] sample (D = 32, 64 or 128) -> power-of-two scales
// 2^exp[p] with |B_jp| 2^exp[p] <= 2^31 - 2^24.  *valid stays false for inf / nan / out-of-range columns.
// Also used by batch_i8.cu for the DATA sample.
pwa_status i8_column_scales(pwa_ctx *ctx, const void *amps, long long n_events, int D, int *exp, float *scale,
                            double *cmax, bool *valid)
{
    *valid = false;
    pwa_status s = ensure_scratch(ctx, 128 * sizeof(unsigned));
    if (s != PWA_OK) return s;
    unsigned *d_cmax = reinterpret_cast<unsigned *>(ctx->d_scratch);
    PWA_CUDA(ctx, cudaMemsetAsync(d_cmax, 0, 128 * sizeof(unsigned), ctx->stream));
    const long long nfloats = n_events * (long long)D;
    long long grid = (nfloats / 4 + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 8;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    i8::k_colmax_f32<<<(unsigned)grid, 256, 0, ctx->stream>>>(reinterpret_cast<const float *>(amps), nfloats, D, d_cmax);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    unsigned h_cmax[128];
    PWA_CUDA(ctx, cudaMemcpyAsync(h_cmax, d_cmax, sizeof(h_cmax), cudaMemcpyDeviceToHost, ctx->stream));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const double qmax = 2147483648.0 - 16777216.0;               // 2^31 - 2^24
    for (int p = 0; p < D; ++p) {
        if (h_cmax[p] >= 0x7f800000u) return PWA_OK;            // inf / nan in the sample: FP64 paths propagate IEEE values
        float c; memcpy(&c, &h_cmax[p], 4);
        int e = 0;
        if (c > 0.0f) {
            e = 30 - ilogbf(c);
            if (ldexp((double)c, e) > qmax) --e;
            if (e > 126) e = 126;
            if (e < -126) return PWA_OK;
        }
        cmax[p] = (double)c;
        for (int g = 0; g < 128 / D; ++g) { exp[g * D + p] = e; scale[g * D + p] = ldexpf(1.0f, e); }
    }
    *valid = true;
    return PWA_OK;
}

// Called after every constant-resonance MC upload: column maxima -> power-of-two scales.
pwa_status prepare_norm_i8(pwa_ctx *ctx)
{
    auto &q = ctx->i8q;
    q.valid = false;
    if (!i8_shape_ok(ctx)) return PWA_OK;
    return i8_column_scales(ctx, ctx->mc.amps, ctx->mc.n_events, 2 * ctx->n, q.exp, q.scale, q.cmax, &q.valid);
}

pwa_status launch_norm_i8(pwa_ctx *ctx, bool *handled, bool three_planes)
{
    *handled = false;
    if (!ctx->i8q.valid || !i8_shape_ok(ctx)) return PWA_OK;
    const int n = ctx->n, D = 2 * n, G = 128 / D;
    const long long N = ctx->mc.n_events;
    const long long rows = N / G;                                // whole 128-real rows
    const int n_tail = (int)(N % G);
    if (rows < 1 || rows > 0x7fffffffLL - i8::TE) return PWA_OK;
    PFN_cuTensorMapEncodeTiled_v12000 enc = tc::tensor_map_encoder();
    if (!enc) return fail(ctx, PWA_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
    alignas(64) CUtensorMap tmap;
    {
        const cuuint64_t gdim[2] = {128, (cuuint64_t)rows};
        const cuuint64_t gstride[1] = {512};
        const cuuint32_t box[2] = {128, (cuuint32_t)i8::TE};
        const cuuint32_t estr[2] = {1, 1};
        CUresult r = enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, ctx->mc.amps, gdim, gstride, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(ctx, PWA_ERR_CUDA, "cuTensorMapEncodeTiled (i8 norm) failed (code " + std::to_string((int)r) + ")");
    }
    const long long ntiles = (rows + i8::TE - 1) / i8::TE;
    long long grid = ctx->sm_count;
    if (grid > ntiles) grid = ntiles;
    static bool s_attr[64] = {false};
    if (!s_attr[ctx->device & 63]) {
        PWA_CUDA(ctx, cudaFuncSetAttribute(i8::k_norm_i8<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)i8::SMEM));
        PWA_CUDA(ctx, cudaFuncSetAttribute(i8::k_norm_i8<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)i8::SMEM));
        s_attr[ctx->device & 63] = true;
    }
    const size_t slot_doubles = (size_t)grid * 16384, dslot_doubles = (size_t)grid * i8::NCW * 128;
    pwa_status s = ensure_scratch(ctx, sizeof(double) * (slot_doubles + 16384 + dslot_doubles + 128));
    if (s != PWA_OK) return s;
    double *slots = reinterpret_cast<double *>(ctx->d_scratch);
    double *ysum = slots + slot_doubles;
    double *dslots = ysum + 16384;
    double *dsum = dslots + dslot_doubles;
    i8::Scales sc;
    i8::Exps ex;
    memcpy(sc.s, ctx->i8q.scale, sizeof(sc.s));
    if (three_planes) for (int p = 0; p < 128; ++p) sc.s[p] = ldexpf(sc.s[p], -8);      // 24 bits below the column maximum
    sc.one = 1;
    memcpy(ex.e, ctx->i8q.exp, sizeof(ex.e));
    if (three_planes) i8::k_norm_i8<3><<<(unsigned)grid, i8::THREADS, i8::SMEM, ctx->stream>>>(tmap, ntiles, sc, slots, dslots);
    else i8::k_norm_i8<4><<<(unsigned)grid, i8::THREADS, i8::SMEM, ctx->stream>>>(tmap, ntiles, sc, slots, dslots);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    i8::k_i8_slot_sum<<<516, 256, 0, ctx->stream>>>(slots, (int)grid, ysum, dslots, dsum);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    const float *tail = reinterpret_cast<const float *>(ctx->mc.amps) + (size_t)rows * 128;
    i8::k_i8_assemble<<<(n * n + 255) / 256, 256, 0, ctx->stream>>>(ysum, dsum, ex, n, tail, n_tail, 1.0 / (double)ctx->mc.n_gen, ctx->d_M, three_planes ? 31 : 24);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    *handled = true;
    return PWA_OK;
}

// A-priori bound on |M_gpu - M_exact|_ab / sqrt(M_aa M_bb)-free absolute form: returns
// max_ab of  N_acc / N_gen * 2 * (eps_q (c_a |B|max_b + c_b |B|max_a) + eps_t c_a c_b),
// with c = 2^(31 - s) per real column (max over re/im of the wave), eps_q = 2^-32, eps_t = 3 * 2^-32 (1 + 2^-7).
// Three planes (M_path == 3): eps_q = 2^-24, eps_t = 2^-23 (1 + 2^-9) (orders t <= 1 dropped: <= (128^2 + 2 * 2^8 * 128^2) 2^-46 c_p c_q).
double norm_i8_error_bound(const pwa_ctx *ctx)
{
    if (!ctx->i8q.valid) return 0.0;
    const int D = 2 * ctx->n;
    double cm = 0.0, bm = 0.0;
    for (int p = 0; p < D; ++p) {
        cm = fmax(cm, ldexp(1.0, 31 - ctx->i8q.exp[p]));
        bm = fmax(bm, ctx->i8q.cmax[p]);
    }
    const bool three = ctx->M_path == 3;
    const double eps_q = three ? ldexp(1.0, -24) : ldexp(1.0, -32);
    const double eps_t = three ? ldexp(1.0, -23) * (1.0 + 1.0 / 512.0) : 3.0 * ldexp(1.0, -32) * (1.0 + 1.0 / 128.0);
    // each complex entry is a sum of two real Gram entries
    return 2.0 * (double)ctx->mc.n_events / (double)ctx->mc.n_gen * (2.0 * eps_q * cm * bm + eps_t * cm * cm);
}

}  // namespace pwa
