// factored.cu — steps A1 + A2-A5 fused (floating masses/widths; BASELINE configs[3]):
// the data pass with the Breit-Wigner factors recomputed in registers from
// (mass_i, Z_{i,s}) — 8 + 16 n_ang bytes per event instead of 16 n — so nothing but the
// factored inputs is read and no amplitude is ever written to HBM.  ALU-bound (fp64).
//
// Mapping: G lanes share an event; lane j owns resonances j, j+G, ... (RPL of them) for all
// angular structures.  Work is done on the dense (resonance x angular structure) grid:
//     S_i   = sum_r BW_r(m_i) * ( sum_s C[r][s] Z_{i,s} ),  C[r][s] = V_wave(r,s) (0 if none)
//     Q[r][s] = sum_i BW_r(m_i) Z_{i,s} / S_i,             T_wave(r,s) = Q[r][s]
// Reduction and finish are shared with data_term.cu (steps A5, A7).
//
// Two-pass floating evaluation (pwa_nll_grad_floating; every evaluation has new masses and widths, so an M built
// for it is used exactly once: the O(N_acc n^2) Gram matrix buys nothing, Norm and its derivatives are O(N_acc n)):
//   RG: the pass also accumulates Q2[r][s] = sum_i BW_r(m_i)^2 Z_{i,s} f_i, from which the host forms
//       U_r = sum_s C[r][s] Q2[r][s] and d/dM_r, d/dG_r (reading A9: dBW/dM = -(2M - iG) BW^2, dBW/dG = i M BW^2);
//   MC: the pass runs over the accepted-MC sample with f_j = conj(S_j) instead of 1 / S_i and no logarithm:
//       component 0 = sum_j |S_j|^2 = N_gen Norm, T'_a = sum_j A_ja conj(S_j) = conj(N_gen (M V)_a)    (eq. 3 second term)
// The record of such a pass is {L or sum|S|^2, n_nonfinite, T[n], Q2[n_res][n_ang]} (complex entries), written through
// the data-term-only output of block_finish (fa.M == nullptr, fa.n = n + n_res n_ang).
#include "factored.cuh"
#include "reduce.cuh"

namespace pwa {

pwa_status fill_fact_args(pwa_ctx *ctx, const Sample &smp, FactArgs *out)
{
    if (!smp.factored) return fail(ctx, PWA_ERR_STATE, "sample is not in factored form");
    if (ctx->res_of_wave.empty()) return fail(ctx, PWA_ERR_STATE, "pwa_set_wave_map not called");
    if (!ctx->res_set) return fail(ctx, PWA_ERR_STATE, "pwa_set_resonances not called");
    if (ctx->n > kMaxFastWaves) return fail(ctx, PWA_ERR_UNSUPPORTED, "factored mode needs n <= 64");
    memset(out, 0, sizeof(*out));
    out->mass = smp.mass;
    out->ang = smp.ang;
    out->n_ang = smp.n_ang;
    out->n_res = ctx->n_res;
    for (int i = 0; i < kMaxRes * kMaxAng; ++i) out->wave_of_pair[i] = -1;
    for (int a = 0; a < ctx->n; ++a) {
        if (ctx->ang_of_wave[a] >= smp.n_ang)
            return fail(ctx, PWA_ERR_INVALID_ARG, "ang_of_wave exceeds the uploaded n_ang");
        out->res_of_wave[a] = (unsigned char)ctx->res_of_wave[a];
        out->ang_of_wave[a] = (unsigned char)ctx->ang_of_wave[a];
        out->wave_of_pair[ctx->res_of_wave[a] * kMaxAng + ctx->ang_of_wave[a]] = (short)a;
    }
    for (int r = 0; r < kMaxRes; ++r) {
        if (r < ctx->n_res) {
            out->rp.m2[r] = ctx->mass0[r] * ctx->mass0[r];
            out->rp.mg[r] = ctx->mass0[r] * ctx->width0[r];
        } else {              // padding resonance: BW ~ 1e-150, coefficient 0
            out->rp.m2[r] = 1e150;
            out->rp.mg[r] = 0.0;
        }
    }
    return PWA_OK;
}

template <typename ST, int G, int RPL, int NANG, int E, int THREADS, bool RG, bool MC>
__global__ void __launch_bounds__(THREADS, 2)
k_data_term_fact(long long N, int n_waves, VArg varg, FactArgs f, FinishArgs fa)
{
    constexpr int GPW = 32 / G, EPB = GPW * E, NWARPS = THREADS / 32;
    constexpr int NQ = RPL * NANG, NACC = RG ? 2 * NQ : NQ;          // accumulators: Q (-> T), then Q2 (-> resonance gradient)
    static_assert(E <= G, "E <= G");
    __shared__ double sV[2 * kMaxFastWaves];
    for (int t = threadIdx.x; t < 2 * n_waves; t += THREADS) sV[t] = varg.v[t];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = lane % G, grp = lane / G;

    double m2r[RPL], mgr[RPL], cr[RPL][NANG], ci[RPL][NANG], qr[NACC], qi[NACC];
#pragma unroll
    for (int rl = 0; rl < RPL; ++rl) {
        const int r = j + G * rl;
        m2r[rl] = f.rp.m2[r]; mgr[rl] = f.rp.mg[r];
#pragma unroll
        for (int s = 0; s < NANG; ++s) {
            const int w = (s < kMaxAng) ? f.wave_of_pair[r * kMaxAng + s] : -1;
            cr[rl][s] = (w >= 0) ? sV[2 * w] : 0.0;
            ci[rl][s] = (w >= 0) ? sV[2 * w + 1] : 0.0;
            qr[rl * NANG + s] = 0.0; qi[rl * NANG + s] = 0.0;
            if (RG) { qr[NQ + rl * NANG + s] = 0.0; qi[NQ + rl * NANG + s] = 0.0; }
        }
    }
    double L = 0.0, bad = 0.0;
    const long long nsteps = (N + EPB - 1) / EPB;
    for (long long b = (long long)blockIdx.x * NWARPS + warp; b < nsteps; b += (long long)gridDim.x * NWARPS) {
        const long long ev0 = b * EPB + (long long)grp * E;
        double2 bw[E][RPL], z[E][NANG];
        double sr[E], si[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const long long ev = ev0 + e;
            const bool valid = ev < N;
            const double m = valid ? __ldg(f.mass + ev) : 0.0;
#pragma unroll
            for (int s = 0; s < NANG; ++s)
                z[e][s] = (valid && s < f.n_ang) ? load_ang<ST>(f.ang, ev, f.n_ang, s) : make_double2(0.0, 0.0);
            sr[e] = 0.0; si[e] = 0.0;
#pragma unroll
            for (int rl = 0; rl < RPL; ++rl) {
                bw[e][rl] = bw_eval(m * m, m2r[rl], mgr[rl]);        // A1
                double wr = 0.0, wi = 0.0;                           // sum_s C[r][s] Z_s
#pragma unroll
                for (int s = 0; s < NANG; ++s) {
                    wr = fma(cr[rl][s], z[e][s].x, wr); wr = fma(-ci[rl][s], z[e][s].y, wr);
                    wi = fma(cr[rl][s], z[e][s].y, wi); wi = fma(ci[rl][s], z[e][s].x, wi);
                }
                sr[e] = fma(bw[e][rl].x, wr, sr[e]); sr[e] = fma(-bw[e][rl].y, wi, sr[e]);   // A2
                si[e] = fma(bw[e][rl].x, wi, si[e]); si[e] = fma(bw[e][rl].y, wr, si[e]);
            }
        }
        // transposing reduction (same scheme as data_term.cu)
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
        for (int m = E; m < G; m <<= 1) { sr[0] += shfl_xor_d(sr[0], m); si[0] += shfl_xor_d(si[0], m); }

        const int my_e = j & (E - 1);
        const bool valid = (ev0 + my_e) < N;
        const double I = sr[0] * sr[0] + si[0] * si[0];
        double rr, rim;
        if (MC) {                                                     // MC pass: f = conj(S), component 0 = sum |S|^2
            rr = sr[0]; rim = -si[0];
            if (valid && j < E) { L += I; if (!isfinite(I)) bad += 1.0; }
        } else {
            const double l = log(I);                                  // A3
            const double inv = 1.0 / I;
            rr = sr[0] * inv; rim = -si[0] * inv;                     // A4: r = 1/S
            if (valid && j < E) { L += l; if (!(I > 0.0) || !isfinite(l)) bad += 1.0; }
        }
        if (!valid) { rr = 0.0; rim = 0.0; }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double er = __shfl_sync(0xffffffffu, rr, e, G);
            const double ei = __shfl_sync(0xffffffffu, rim, e, G);
#pragma unroll
            for (int s = 0; s < NANG; ++s) {
                const double gr = z[e][s].x * er - z[e][s].y * ei;    // Z_s r_i
                const double gi = z[e][s].x * ei + z[e][s].y * er;
#pragma unroll
                for (int rl = 0; rl < RPL; ++rl) {
                    qr[rl * NANG + s] = fma(bw[e][rl].x, gr, qr[rl * NANG + s]); qr[rl * NANG + s] = fma(-bw[e][rl].y, gi, qr[rl * NANG + s]);
                    qi[rl * NANG + s] = fma(bw[e][rl].x, gi, qi[rl * NANG + s]); qi[rl * NANG + s] = fma(bw[e][rl].y, gr, qi[rl * NANG + s]);
                    if (RG) {                                         // A9: the same with BW^2
                        const double b2r = fma(bw[e][rl].x, bw[e][rl].x, -bw[e][rl].y * bw[e][rl].y), b2i = 2.0 * bw[e][rl].x * bw[e][rl].y;
                        qr[NQ + rl * NANG + s] = fma(b2r, gr, qr[NQ + rl * NANG + s]); qr[NQ + rl * NANG + s] = fma(-b2i, gi, qr[NQ + rl * NANG + s]);
                        qi[NQ + rl * NANG + s] = fma(b2r, gi, qi[NQ + rl * NANG + s]); qi[NQ + rl * NANG + s] = fma(b2i, gr, qi[NQ + rl * NANG + s]);
                    }
                }
            }
        }
    }
    // accumulator idx -> component of the record: Q[r][s] -> wave(r, s); Q2[r][s] -> n + r n_ang + s
    auto wave_of = [&](int idx) -> int {
        const int base = idx % NQ, rl = base / NANG, s = base % NANG, r = j + G * rl;
        if (idx < NQ) return (s < kMaxAng) ? (int)f.wave_of_pair[r * kMaxAng + s] : -1;
        return (r < f.n_res && s < f.n_ang) ? n_waves + r * f.n_ang + s : -1;
    };
    reduce_and_finish<G, NACC, THREADS>(L, bad, qr, qi, wave_of, sV, fa);
}

// mode 0: plain data pass; 1: data pass + resonance-gradient sums; 2: MC pass (Norm, its V gradient, resonance-gradient sums)
template <typename ST, int G, int RPL, int NANG, int E>
static pwa_status launch_fact(pwa_ctx *ctx, const VArg &varg, const FactArgs &f, const FinishArgs &fa_in, int mode, long long N)
{
    constexpr int THREADS = 256, EPB = (32 / G) * E, NWARPS = THREADS / 32;
    auto kern = mode == 0 ? k_data_term_fact<ST, G, RPL, NANG, E, THREADS, false, false>
              : mode == 1 ? k_data_term_fact<ST, G, RPL, NANG, E, THREADS, true, false>
                          : k_data_term_fact<ST, G, RPL, NANG, E, THREADS, true, true>;
    int occ = 0;
    PWA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    long long nsteps = (N + EPB - 1) / EPB, want = (nsteps + NWARPS - 1) / NWARPS;
    long long grid = (long long)ctx->sm_count * occ;
    if (want < grid) grid = want;
    if (grid < 1) grid = 1;
    FinishArgs fa = fa_in;
    pwa_status s = ensure_partials(ctx, (size_t)n_components(fa.n) * (size_t)grid);
    if (s != PWA_OK) return s;
    fa.partials = ctx->d_partials;
    kern<<<(unsigned)grid, THREADS, 0, ctx->stream>>>(N, ctx->n, varg, f, fa);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

template <typename ST, int NANG>
static pwa_status dispatch_fact(pwa_ctx *ctx, const VArg &varg, const FactArgs &f, const FinishArgs &fa, int mode, long long N)
{
    const int nr = ctx->n_res;
    if (nr <= 4)  return launch_fact<ST, 4, 1, NANG, 4>(ctx, varg, f, fa, mode, N);
    if (nr <= 8)  return launch_fact<ST, 4, 2, NANG, 4>(ctx, varg, f, fa, mode, N);
    if (nr <= 16) return launch_fact<ST, 8, 2, NANG, 4>(ctx, varg, f, fa, mode, N);
    if (nr <= 32) return launch_fact<ST, 8, 4, NANG, 2>(ctx, varg, f, fa, mode, N);
    return launch_fact<ST, 16, 4, NANG, 2>(ctx, varg, f, fa, mode, N);
}

static pwa_status run_fact_pass(pwa_ctx *ctx, const Sample &smp, const double *Vk, const FinishArgs &fa, int mode)
{
    FactArgs f;
    pwa_status s = fill_fact_args(ctx, smp, &f);
    if (s != PWA_OK) return s;
    VArg varg;
    memset(&varg, 0, sizeof(varg));
    for (int t = 0; t < 2 * ctx->n; ++t) varg.v[t] = Vk[t];
    const bool f32 = ctx->storage == PWA_F32;
    if (smp.n_ang <= 2)
        return f32 ? dispatch_fact<float, 2>(ctx, varg, f, fa, mode, smp.n_events) : dispatch_fact<double, 2>(ctx, varg, f, fa, mode, smp.n_events);
    return f32 ? dispatch_fact<float, 4>(ctx, varg, f, fa, mode, smp.n_events) : dispatch_fact<double, 4>(ctx, varg, f, fa, mode, smp.n_events);
}

pwa_status launch_factored_data_term(pwa_ctx *ctx, const double *Vk, const FinishArgs &fa)
{
    return run_fact_pass(ctx, ctx->data, Vk, fa, 0);
}

// Two-pass floating evaluation: the MC pass (record k = 0) and the data pass (record k = 1), each with the
// resonance-gradient sums, written as data-term-only records of n + n_res n_ang complex components into the mapped
// result area; flags 0 and 1 are raised when the records are complete.  Needs n + n_res * n_ang <= 64 (the block
// reduction holds 2 + 2 * 64 components) and equal n_ang of the two samples.
pwa_status launch_floating_passes(pwa_ctx *ctx, const double *V, int *ncomp_out)
{
    const int n_ext = ctx->n + ctx->n_res * ctx->data.n_ang;
    if (n_ext > kMaxFastWaves || ctx->data.n_ang != ctx->mc.n_ang)
        return fail(ctx, PWA_ERR_UNSUPPORTED, "two-pass floating evaluation needs n + n_res * n_ang <= 64 and equal n_ang");
    const int NC = n_components(n_ext);
    *ncomp_out = NC;
    ++ctx->seq;
    for (int k = 0; k < 2; ++k) {
        FinishArgs fa;
        fa.partials = nullptr; fa.ticket = ctx->d_ticket; fa.M = nullptr; fa.n = n_ext;
        fa.out = ctx->dev_result + (size_t)k * NC;
        fa.done_flag = ctx->dev_flags + k; fa.seq = ctx->seq;
        pwa_status s = run_fact_pass(ctx, k == 0 ? ctx->mc : ctx->data, V, fa, k == 0 ? 2 : 1);
        if (s != PWA_OK) return s;
    }
    ctx->last_K = 0;                              // the records are not evaluation records: pwa_fetch must not read them
    return PWA_OK;
}

}  // namespace pwa
