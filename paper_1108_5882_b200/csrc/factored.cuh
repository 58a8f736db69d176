// factored.cuh — step A1 (with floating masses/widths nothing can be pre-calculated):
// amplitudes are rebuilt on the fly as
//     A_ia = BW(m_i; M_r(a), G_r(a)) * Z_{i,s(a)},   BW(m; M, G) = 1 / (M^2 - m^2 - i M G)   (C3)
// from the per-event mass and the precomputed angular factors Z.
#pragma once
#include <cuda_runtime.h>
#include <string.h>

#include "pwa_internal.h"

namespace pwa {

struct FactArgs {                         // by-value kernel argument (~2.3 KB)
    const double *mass;                   // [N]
    const void *ang;                      // [N][n_ang] complex, storage type
    int n_ang, n_res;
    unsigned char res_of_wave[kMaxFastWaves];
    unsigned char ang_of_wave[kMaxFastWaves];
    short wave_of_pair[kMaxRes * kMaxAng];  // (r, s) -> wave or -1
    ResParams rp;                         // M_r^2 and M_r G_r; padded resonances: m2 = 1e300
};

__device__ __forceinline__ double2 bw_eval(double m2, double M2, double MG)
{
    // 1/(d - i MG) = (d + i MG) / (d^2 + MG^2),  d = M^2 - m^2
    const double d = M2 - m2;
    const double inv = 1.0 / fma(d, d, MG * MG);
    return make_double2(d * inv, MG * inv);
}

// 1/x for normal positive x: MUFU.RCP64H seed + two Newton steps (<= ~1 ulp); anything else
// (0, denormal, inf, nan, negative) takes the IEEE division.
__device__ __forceinline__ double rcp_pos(double x)
{
    const unsigned ex = ((unsigned)__double2hiint(x) >> 20) & 0xfffu;   // sign + biased exponent
    if (ex - 1u >= 0x7feu) return 1.0 / x;
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

__device__ __forceinline__ double2 bw_eval_fast(double m2, double M2, double MG)
{
    const double d = M2 - m2;
    const double inv = rcp_pos(fma(d, d, MG * MG));
    return make_double2(d * inv, MG * inv);
}

// one complex angular factor, one vector load (the array is 16-byte aligned: upload contract)
template <typename ST>
__device__ __forceinline__ double2 load_ang(const void *ang, long long ev, int n_ang, int s)
{
    if (sizeof(ST) == 8) {
        return __ldg(reinterpret_cast<const double2 *>(ang) + (ev * n_ang + s));
    } else {
        const float2 z = __ldg(reinterpret_cast<const float2 *>(ang) + (ev * n_ang + s));
        return make_double2((double)z.x, (double)z.y);
    }
}

template <typename ST>
__device__ __forceinline__ double2 factored_amp(const FactArgs &f, long long ev, int a)
{
    const double m = f.mass[ev];
    const int r = f.res_of_wave[a], s = f.ang_of_wave[a];
    const double2 bw = bw_eval(m * m, f.rp.m2[r], f.rp.mg[r]);
    const double2 z = load_ang<ST>(f.ang, ev, f.n_ang, s);
    return make_double2(bw.x * z.x - bw.y * z.y, bw.x * z.y + bw.y * z.x);
}

pwa_status fill_fact_args(pwa_ctx *ctx, const Sample &smp, FactArgs *out);

}  // namespace pwa
