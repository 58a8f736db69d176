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

template <typename ST, int G, int RPL, int NANG, int E, int THREADS>
__global__ void __launch_bounds__(THREADS, 2)
k_data_term_fact(long long N, VArg varg, FactArgs f, FinishArgs fa)
{
    constexpr int GPW = 32 / G, EPB = GPW * E, NWARPS = THREADS / 32;
    static_assert(E <= G, "E <= G");
    __shared__ double sV[2 * kMaxFastWaves];
    for (int t = threadIdx.x; t < 2 * fa.n; t += THREADS) sV[t] = varg.v[t];
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = lane % G, grp = lane / G;

    double m2r[RPL], mgr[RPL], cr[RPL][NANG], ci[RPL][NANG], qr[RPL * NANG], qi[RPL * NANG];
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
        const double l = log(I);                                      // A3
        const double inv = 1.0 / I;
        double rr = sr[0] * inv, rim = -si[0] * inv;                  // A4: r = 1/S
        if (valid && j < E) { L += l; if (!(I > 0.0) || !isfinite(l)) bad += 1.0; }
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
                }
            }
        }
    }
    auto wave_of = [&](int idx) -> int {
        const int rl = idx / NANG, s = idx % NANG;
        return (s < kMaxAng) ? (int)f.wave_of_pair[(j + G * rl) * kMaxAng + s] : -1;
    };
    reduce_and_finish<G, RPL * NANG, THREADS>(L, bad, qr, qi, wave_of, sV, fa);
}

template <typename ST, int G, int RPL, int NANG, int E>
static pwa_status launch_fact(pwa_ctx *ctx, const VArg &varg, const FactArgs &f, const FinishArgs &fa_in)
{
    constexpr int THREADS = 256, EPB = (32 / G) * E, NWARPS = THREADS / 32;
    auto kern = k_data_term_fact<ST, G, RPL, NANG, E, THREADS>;
    int occ = 0;
    PWA_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, THREADS, 0));
    if (occ < 1) occ = 1;
    const long long N = ctx->data.n_events;
    long long nsteps = (N + EPB - 1) / EPB, want = (nsteps + NWARPS - 1) / NWARPS;
    long long grid = (long long)ctx->sm_count * occ;
    if (want < grid) grid = want;
    if (grid < 1) grid = 1;
    FinishArgs fa = fa_in;
    pwa_status s = ensure_partials(ctx, (size_t)n_components(ctx->n) * (size_t)grid);
    if (s != PWA_OK) return s;
    fa.partials = ctx->d_partials;
    kern<<<(unsigned)grid, THREADS, 0, ctx->stream>>>(N, varg, f, fa);
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

template <typename ST, int NANG>
static pwa_status dispatch_fact(pwa_ctx *ctx, const VArg &varg, const FactArgs &f, const FinishArgs &fa)
{
    const int nr = ctx->n_res;
    if (nr <= 4)  return launch_fact<ST, 4, 1, NANG, 4>(ctx, varg, f, fa);
    if (nr <= 8)  return launch_fact<ST, 4, 2, NANG, 4>(ctx, varg, f, fa);
    if (nr <= 16) return launch_fact<ST, 8, 2, NANG, 4>(ctx, varg, f, fa);
    if (nr <= 32) return launch_fact<ST, 8, 4, NANG, 2>(ctx, varg, f, fa);
    return launch_fact<ST, 16, 4, NANG, 2>(ctx, varg, f, fa);
}

pwa_status launch_factored_data_term(pwa_ctx *ctx, const double *Vk, const FinishArgs &fa)
{
    FactArgs f;
    pwa_status s = fill_fact_args(ctx, ctx->data, &f);
    if (s != PWA_OK) return s;
    VArg varg;
    memset(&varg, 0, sizeof(varg));
    for (int t = 0; t < 2 * ctx->n; ++t) varg.v[t] = Vk[t];
    const bool f32 = ctx->storage == PWA_F32;
    if (ctx->data.n_ang <= 2)
        return f32 ? dispatch_fact<float, 2>(ctx, varg, f, fa) : dispatch_fact<double, 2>(ctx, varg, f, fa);
    return f32 ? dispatch_fact<float, 4>(ctx, varg, f, fa) : dispatch_fact<double, 4>(ctx, varg, f, fa);
}

}  // namespace pwa
