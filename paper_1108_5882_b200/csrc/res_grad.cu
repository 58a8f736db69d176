// res_grad.cu — reading A9 (extension; the paper discusses only the V parameters but fits
// with floating masses/widths, need these derivatives):
//   d_theta S_i = w_{r,i} d_theta BW_r(m_i),   w_{r,i} = sum_{a: r(a)=r} V_a Z_{i,s(a)}
//   dBW/dM = -(2M - iG) BW^2,  dBW/dG = i M BW^2                                  (C3)
//   d L_data / d theta = 2 sum_i Re( d_theta S_i / S_i )
//   d Norm   / d theta = (2/N_gen) sum_j Re( conj(S_j) d_theta S_j )
// The event-independent factors are pulled out: one complex accumulator per resonance,
//   U_r = sum_i w_{r,i} BW_r(m_i)^2 * f_i,   f_i = 1/S_i (data) or conj(S_i) (MC),
// and the host applies -(2M - iG) and iM.  Thread per event; warp + block tree as in A5.
// The MC pass also sums |S_j|^2 (component 0 of its record): Norm = sum_j |S_j|^2 / N_gen at the CURRENT resonance
// parameters, which the eq. 2 form needs (d nll2 / d theta = -d L_data + (N_data / Norm) d Norm, reading C2).
#include "factored.cuh"
#include "reduce.cuh"

namespace pwa {

constexpr int RG_THREADS = 128;

template <typename ST>
__global__ void __launch_bounds__(RG_THREADS)
k_res_grad(long long N, int mode, int n, VArg varg, FactArgs f, FinishArgs fa)
{
    constexpr int NWARPS = RG_THREADS / 32;
    __shared__ double sV[2 * kMaxFastWaves];
    __shared__ double2 sC[kMaxRes * kMaxAng];
    __shared__ double s_acc[NWARPS][2 + 2 * kMaxRes];
    __shared__ double s_tot[2 + 2 * kMaxRes];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_res = f.n_res, n_ang = f.n_ang, NC = 2 + 2 * n_res;
    for (int t = tid; t < 2 * n; t += RG_THREADS) sV[t] = varg.v[t];
    __syncthreads();
    for (int t = tid; t < n_res * kMaxAng; t += RG_THREADS) {
        const int w = f.wave_of_pair[t];
        sC[t] = (w >= 0) ? make_double2(sV[2 * w], sV[2 * w + 1]) : make_double2(0.0, 0.0);
    }
    for (int t = tid; t < NWARPS * (2 + 2 * kMaxRes); t += RG_THREADS) (&s_acc[0][0])[t] = 0.0;
    __syncthreads();
    const long long stride = (long long)gridDim.x * RG_THREADS;
    const long long nround = (N + stride - 1) / stride;
    for (long long it = 0; it < nround; ++it) {
        const long long i = it * stride + (long long)blockIdx.x * RG_THREADS + tid;
        const bool valid = i < N;
        const long long ev = valid ? i : 0;
        const double m = f.mass[ev], mm = m * m;
        double2 z[kMaxAng];
#pragma unroll
        for (int s = 0; s < kMaxAng; ++s) z[s] = (s < n_ang) ? load_ang<ST>(f.ang, ev, n_ang, s) : make_double2(0.0, 0.0);
        double sr = 0.0, si = 0.0;
        for (int r = 0; r < n_res; ++r) {
            const double2 bw = bw_eval(mm, f.rp.m2[r], f.rp.mg[r]);
            double wr = 0.0, wi = 0.0;
#pragma unroll
            for (int s = 0; s < kMaxAng; ++s) {
                const double2 c = sC[r * kMaxAng + s];
                wr += c.x * z[s].x - c.y * z[s].y; wi += c.x * z[s].y + c.y * z[s].x;
            }
            sr += bw.x * wr - bw.y * wi; si += bw.x * wi + bw.y * wr;
        }
        double fr, fi;
        if (mode == 0) { const double inv = 1.0 / (sr * sr + si * si); fr = sr * inv; fi = -si * inv; }
        else           { fr = sr; fi = -si; }
        if (!valid) { fr = 0.0; fi = 0.0; }
        if (mode == 1) {                         // uniform branch
            const double i2 = warp_sum(valid ? sr * sr + si * si : 0.0);
            if (lane == 0) s_acc[warp][0] += i2;
        }
        for (int r = 0; r < n_res; ++r) {
            const double2 bw = bw_eval(mm, f.rp.m2[r], f.rp.mg[r]);
            double wr = 0.0, wi = 0.0;
#pragma unroll
            for (int s = 0; s < kMaxAng; ++s) {
                const double2 c = sC[r * kMaxAng + s];
                wr += c.x * z[s].x - c.y * z[s].y; wi += c.x * z[s].y + c.y * z[s].x;
            }
            const double b2r = bw.x * bw.x - bw.y * bw.y, b2i = 2.0 * bw.x * bw.y;
            const double pr = wr * b2r - wi * b2i, pi = wr * b2i + wi * b2r;
            double ur = pr * fr - pi * fi, ui = pr * fi + pi * fr;
            ur = warp_sum(ur); ui = warp_sum(ui);
            if (lane == 0) { s_acc[warp][2 + 2 * r] += ur; s_acc[warp][3 + 2 * r] += ui; }
        }
    }
    __syncthreads();
    for (int c = tid; c < NC; c += RG_THREADS) {
        double t = 0.0;
        for (int w = 0; w < NWARPS; ++w) t += s_acc[w][c];
        s_tot[c] = t;
    }
    __syncthreads();
    block_finish(s_tot, &s_acc[0][0], sV, fa);
}

// Same sums for n_res <= NR, n_ang <= NA (configs[3]: 8 resonances x 2 angular structures): every Breit-Wigner is
// evaluated once per event and kept in registers, the per-resonance sums U_r stay in per-thread fp64 registers for
// the thread's whole event range and meet the warp / block tree only once at the end (the generic kernel above
// pays two warp reductions per resonance and event round).  fp64-ALU bound: ~450 fp64 instructions per event.
template <typename ST, int NR, int NA>
__global__ void __launch_bounds__(RG_THREADS)
k_res_grad_fast(long long N, int mode, int n, VArg varg, FactArgs f, FinishArgs fa)
{
    constexpr int NWARPS = RG_THREADS / 32;
    __shared__ double sV[2 * kMaxFastWaves];
    __shared__ double2 sC[NR * NA];
    __shared__ double s_acc[NWARPS][2 + 2 * NR];
    __shared__ double s_tot[2 + 2 * kMaxRes];
    __shared__ double s_red[RG_THREADS];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_res = f.n_res, n_ang = f.n_ang, NC = 2 + 2 * n_res;
    for (int t = tid; t < 2 * n; t += RG_THREADS) sV[t] = varg.v[t];
    __syncthreads();
    for (int t = tid; t < NR * NA; t += RG_THREADS) {
        const int r = t / NA, sg = t % NA;
        const int w = (r < n_res && sg < n_ang) ? f.wave_of_pair[r * kMaxAng + sg] : -1;
        sC[t] = (w >= 0) ? make_double2(sV[2 * w], sV[2 * w + 1]) : make_double2(0.0, 0.0);
    }
    __syncthreads();
    double ur[NR], ui[NR];
#pragma unroll
    for (int r = 0; r < NR; ++r) { ur[r] = 0.0; ui[r] = 0.0; }
    double i2 = 0.0;                             // MC pass: sum_j |S_j|^2
    const long long stride = (long long)gridDim.x * RG_THREADS;
    for (long long i = (long long)blockIdx.x * RG_THREADS + tid; i < N; i += stride) {
        const double m = __ldg(f.mass + i), mm = m * m;
        double2 z[NA];
#pragma unroll
        for (int sg = 0; sg < NA; ++sg) z[sg] = (sg < n_ang) ? load_ang<ST>(f.ang, i, n_ang, sg) : make_double2(0.0, 0.0);
        double pr[NR], pi[NR];                   // w_r BW_r^2
        double sr = 0.0, si = 0.0;
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            const double2 bw = r < n_res ? bw_eval_fast(mm, f.rp.m2[r], f.rp.mg[r]) : make_double2(0.0, 0.0);
            double wr = 0.0, wi = 0.0;
#pragma unroll
            for (int sg = 0; sg < NA; ++sg) {
                const double2 c = sC[r * NA + sg];
                wr = fma(c.x, z[sg].x, wr); wr = fma(-c.y, z[sg].y, wr);
                wi = fma(c.x, z[sg].y, wi); wi = fma(c.y, z[sg].x, wi);
            }
            const double tr = bw.x * wr - bw.y * wi, ti = bw.x * wi + bw.y * wr;   // w BW
            sr += tr; si += ti;
            pr[r] = tr * bw.x - ti * bw.y; pi[r] = tr * bw.y + ti * bw.x;           // w BW^2
        }
        double fr, fi;
        if (mode == 0) { const double inv = 1.0 / (sr * sr + si * si); fr = sr * inv; fi = -si * inv; }
        else           { fr = sr; fi = -si; i2 = fma(sr, sr, i2); i2 = fma(si, si, i2); }
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            ur[r] = fma(pr[r], fr, ur[r]); ur[r] = fma(-pi[r], fi, ur[r]);
            ui[r] = fma(pr[r], fi, ui[r]); ui[r] = fma(pi[r], fr, ui[r]);
        }
    }
#pragma unroll
    for (int r = 0; r < NR; ++r) {
        const double a = warp_sum(ur[r]), b = warp_sum(ui[r]);
        if (lane == 0) { s_acc[warp][2 + 2 * r] = a; s_acc[warp][3 + 2 * r] = b; }
    }
    i2 = warp_sum(i2);
    if (lane == 0) { s_acc[warp][0] = i2; s_acc[warp][1] = 0.0; }
    __syncthreads();
    for (int c = tid; c < NC; c += RG_THREADS) {
        double t = 0.0;
        for (int w = 0; w < NWARPS; ++w) t += s_acc[w][c];
        s_tot[c] = t;
    }
    __syncthreads();
    block_finish(s_tot, s_red, sV, fa);
}

static pwa_status run_pass(pwa_ctx *ctx, const Sample &smp, int mode, const VArg &varg, double *out_dev)
{
    FactArgs f;
    pwa_status s = fill_fact_args(ctx, smp, &f);
    if (s != PWA_OK) return s;
    const long long N = smp.n_events;
    long long grid = (N + RG_THREADS - 1) / RG_THREADS;
    const long long cap = (long long)ctx->sm_count * 8;
    if (grid > cap) grid = cap;
    if (grid < 1) grid = 1;
    const int NC = 2 + 2 * ctx->n_res;
    s = ensure_partials(ctx, (size_t)NC * (size_t)grid);
    if (s != PWA_OK) return s;
    FinishArgs fa;
    fa.partials = ctx->d_partials; fa.ticket = ctx->d_ticket; fa.M = nullptr; fa.out = out_dev; fa.n = ctx->n_res;
    const bool fast = ctx->n_res <= 8 && smp.n_ang <= 2 && ctx->opt_data_term != 99;
    if (fast) {
        if (ctx->storage == PWA_F32) k_res_grad_fast<float, 8, 2><<<(unsigned)grid, RG_THREADS, 0, ctx->stream>>>(N, mode, ctx->n, varg, f, fa);
        else                         k_res_grad_fast<double, 8, 2><<<(unsigned)grid, RG_THREADS, 0, ctx->stream>>>(N, mode, ctx->n, varg, f, fa);
    } else {
        if (ctx->storage == PWA_F32) k_res_grad<float><<<(unsigned)grid, RG_THREADS, 0, ctx->stream>>>(N, mode, ctx->n, varg, f, fa);
        else                         k_res_grad<double><<<(unsigned)grid, RG_THREADS, 0, ctx->stream>>>(N, mode, ctx->n, varg, f, fa);
    }
    ctx->launches++;
    PWA_CUDA(ctx, cudaGetLastError());
    return PWA_OK;
}

pwa_status launch_res_grad(pwa_ctx *ctx, const double *V, double *dM, double *dG)
{
    const int nr = ctx->n_res, NC = 2 + 2 * nr;
    VArg varg;
    memset(&varg, 0, sizeof(varg));
    for (int t = 0; t < 2 * ctx->n; ++t) varg.v[t] = V[t];
    double *dev = ctx->d_result;            // [2][NC] scratch records
    pwa_status s = run_pass(ctx, ctx->data, 0, varg, dev);
    if (s != PWA_OK) return s;
    s = run_pass(ctx, ctx->mc, 1, varg, dev + NC);
    if (s != PWA_OK) return s;
    PWA_CUDA(ctx, cudaMemcpyAsync(ctx->h_result, dev, sizeof(double) * 2 * NC, cudaMemcpyDeviceToHost, ctx->stream));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->last_K = 0;
    const double *Ud = ctx->h_result + 2, *Um = ctx->h_result + NC + 2;
    const double inv_ngen = 1.0 / (double)ctx->mc.n_gen;
    // eq. 3: nll = -L_data + Norm;  eq. 2 ("likelihood" = 1): nll2 = -L_data + N_data ln Norm, so the Norm part of the
    // derivative carries N_data / Norm (Norm from the MC pass itself: valid for the current resonance parameters)
    const double norm_now = ctx->h_result[NC] * inv_ngen;
    const double wN = ctx->opt_likelihood == 1 ? eq2_n_data(ctx) / norm_now : 1.0;
    for (int r = 0; r < nr; ++r) {
        const double M = ctx->mass0[r], G = ctx->width0[r];
        // Re( -(2M - iG) U ) = -(2M Ur + G Ui) ;  Re( iM U ) = -M Ui
        const double dL_dM = 2.0 * (-(2.0 * M * Ud[2 * r] + G * Ud[2 * r + 1]));
        const double dL_dG = 2.0 * (-M * Ud[2 * r + 1]);
        const double dN_dM = 2.0 * inv_ngen * (-(2.0 * M * Um[2 * r] + G * Um[2 * r + 1]));
        const double dN_dG = 2.0 * inv_ngen * (-M * Um[2 * r + 1]);
        dM[r] = -dL_dM + wN * dN_dM;
        dG[r] = -dL_dG + wN * dN_dG;
    }
    return PWA_OK;
}

}  // namespace pwa
