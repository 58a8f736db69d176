/*
 * synth_gen.c — seeded synthetic INPUT generator (shared by the oracle tests, the CUDA
 * parity tests and bench.py).  It produces the arrays both sides consume; it holds none of
 * the likelihood/gradient arithmetic of the method and is not linked into libpwa.so nor
 * into the oracle.  The recipe follows BASELINE.json configs[0..4] and DESIGN.md section 4
 * (readings C4, C5, C9-C13, C15).  The real BES J/psi -> gamma K+K- sample is NOT
 * reconstructed: these events only have its shape (events x waves complex amplitudes that
 * are Breit-Wigner x spherical-harmonic products; accepted phase-space MC).
 *
 * RNG (C15): counter based, order independent:
 *     u64(seed, stream, ctr) = mix(mix(mix(seed) ^ mix(stream)) + ctr * GOLDEN)
 * so any thread count / chunking yields the identical arrays.
 *
 * Kinematics (C12): m ~ U[0.988, 3.0] GeV, cos(theta) ~ U[-1, 1], phi ~ U[0, 2pi).
 * Candidate c of a sample with base stream s0 uses (s0, c) for m, (s0+1, c) for cos,
 * (s0+2, c) for phi and (s0+3, c) for the accept/reject uniform.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define M_LO 0.988
#define M_HI 3.0
#define TWO_PI 6.283185307179586476925286766559

static inline uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t pwa_gen_u64(uint64_t seed, uint64_t stream, uint64_t ctr)
{
    uint64_t key = mix64(mix64(seed) ^ mix64(stream));
    return mix64(key + ctr * 0x9E3779B97F4A7C15ULL);
}

static inline double u01(uint64_t seed, uint64_t stream, uint64_t ctr)
{
    return (double)(pwa_gen_u64(seed, stream, ctr) >> 11) * (1.0 / 9007199254740992.0);
}

void pwa_gen_uniform(uint64_t seed, uint64_t stream, int64_t start, int64_t count,
                     double lo, double hi, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < count; ++k)
        out[k] = lo + (hi - lo) * u01(seed, stream, (uint64_t)(start + k));
}

/* complex standard normal (C13): Re, Im independent N(0,1), Box-Muller. out: [count][2] */
void pwa_gen_cnormal(uint64_t seed, uint64_t stream, int64_t start, int64_t count, double *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < count; ++k) {
        double u1 = u01(seed, stream, (uint64_t)(2 * (start + k)));
        double u2 = u01(seed, stream, (uint64_t)(2 * (start + k) + 1));
        double r = sqrt(-2.0 * log(1.0 - u1));
        out[2 * k]     = r * cos(TWO_PI * u2);
        out[2 * k + 1] = r * sin(TWO_PI * u2);
    }
}

/* Angular structures (C4), Condon-Shortley: id 0: Y00, 1: Y20, 2: Y2+1, 3: Y2-1 */
static inline void ylm(int id, double c, double phi, double *re, double *im)
{
    double s = sqrt(fmax(0.0, 1.0 - c * c));
    switch (id) {
    case 0: *re = 0.28209479177387814; *im = 0.0; break;
    case 1: *re = 0.31539156525252005 * (3.0 * c * c - 1.0); *im = 0.0; break;
    case 2: { double k = -0.7725484040463791 * s * c; *re = k * cos(phi); *im = k * sin(phi); } break;
    default: { double k = 0.7725484040463791 * s * c; *re = k * cos(phi); *im = -k * sin(phi); } break;
    }
}

/* generator's own resonance line shape (C3): 1 / (M^2 - m^2 - i M G) */
static inline void lineshape(double m, double M, double G, double *re, double *im)
{
    double a = M * M - m * m, b = M * G;
    double d = a * a + b * b;
    *re = a / d; *im = b / d;
}

static inline double efficiency(double m, double c) { (void)m; return 0.6 + 0.3 * c * c; }

static double intensity_at(double m, double c, double phi, int n_res, const double *Mr,
                           const double *Gr, int n, const int32_t *res_of_wave,
                           const int32_t *yid_of_wave, const double *V, double *bwbuf)
{
    double yr[4], yi[4];
    for (int k = 0; k < 4; ++k) ylm(k, c, phi, &yr[k], &yi[k]);
    for (int r = 0; r < n_res; ++r) lineshape(m, Mr[r], Gr[r], &bwbuf[2 * r], &bwbuf[2 * r + 1]);
    double sr = 0.0, si = 0.0;
    for (int a = 0; a < n; ++a) {
        int r = res_of_wave[a], y = yid_of_wave[a];
        double ar = bwbuf[2 * r] * yr[y] - bwbuf[2 * r + 1] * yi[y];
        double ai = bwbuf[2 * r] * yi[y] + bwbuf[2 * r + 1] * yr[y];
        sr += V[2 * a] * ar - V[2 * a + 1] * ai;
        si += V[2 * a] * ai + V[2 * a + 1] * ar;
    }
    return sr * sr + si * si;
}

/* max over a pilot of `count` uniform candidates of (eff *) I  (C11) */
double pwa_gen_pilot_max(uint64_t seed, uint64_t s0, int64_t count, int use_eff, int n_res,
                         const double *Mr, const double *Gr, int n, const int32_t *res_of_wave,
                         const int32_t *yid_of_wave, const double *V)
{
    double best = 0.0;
#pragma omp parallel
    {
        double *bw = (double *)malloc(sizeof(double) * 2 * (size_t)n_res);
        double loc = 0.0;
#pragma omp for schedule(static)
        for (int64_t k = 0; k < count; ++k) {
            double m = M_LO + (M_HI - M_LO) * u01(seed, s0, (uint64_t)k);
            double c = -1.0 + 2.0 * u01(seed, s0 + 1, (uint64_t)k);
            double p = TWO_PI * u01(seed, s0 + 2, (uint64_t)k);
            double I = intensity_at(m, c, p, n_res, Mr, Gr, n, res_of_wave, yid_of_wave, V, bw);
            if (use_eff) I *= efficiency(m, c);
            if (I > loc) loc = I;
        }
#pragma omp critical
        { if (loc > best) best = loc; }
        free(bw);
    }
    return best;
}

/* Accept/reject in candidate-index order until n_want events are accepted.
 * mode bit0: multiply by efficiency eps(m, cos) (C10); bit1: multiply by I(Omega)/I_max.
 * mode 0: every candidate accepted (cfg 0 MC).  Returns the number accepted (== n_want);
 * *n_drawn = index of the last accepted candidate + 1 (C9: N_gen for MC samples);
 * *n_over  = candidates with weight > 1 (C11; expected 0). */
int64_t pwa_gen_accept(uint64_t seed, uint64_t s0, int64_t n_want, int mode, double I_max,
                       int n_res, const double *Mr, const double *Gr, int n,
                       const int32_t *res_of_wave, const int32_t *yid_of_wave, const double *V,
                       double *m_out, double *c_out, double *p_out, int64_t *n_drawn,
                       int64_t *n_over)
{
    const int64_t CH = 1 << 21;
    double *mm = (double *)malloc(sizeof(double) * CH);
    double *cc = (double *)malloc(sizeof(double) * CH);
    double *pp = (double *)malloc(sizeof(double) * CH);
    uint8_t *fl = (uint8_t *)malloc(CH);
    int64_t got = 0, base = 0, over = 0, last = -1;
    while (got < n_want) {
        int64_t ov = 0;
#pragma omp parallel reduction(+ : ov)
        {
            double *bw = (double *)malloc(sizeof(double) * 2 * (size_t)(n_res > 0 ? n_res : 1));
#pragma omp for schedule(static)
            for (int64_t k = 0; k < CH; ++k) {
                uint64_t c = (uint64_t)(base + k);
                double m = M_LO + (M_HI - M_LO) * u01(seed, s0, c);
                double ct = -1.0 + 2.0 * u01(seed, s0 + 1, c);
                double ph = TWO_PI * u01(seed, s0 + 2, c);
                double w = 1.0;
                if (mode & 1) w *= efficiency(m, ct);
                if (mode & 2)
                    w *= intensity_at(m, ct, ph, n_res, Mr, Gr, n, res_of_wave, yid_of_wave, V, bw) / I_max;
                if (w > 1.0) ov += 1;
                mm[k] = m; cc[k] = ct; pp[k] = ph;
                fl[k] = (mode == 0) ? 1 : (u01(seed, s0 + 3, c) < w);
            }
            free(bw);
        }
        over += ov;
        for (int64_t k = 0; k < CH && got < n_want; ++k)
            if (fl[k]) {
                m_out[got] = mm[k]; c_out[got] = cc[k]; p_out[got] = pp[k];
                last = base + k; ++got;
            }
        base += CH;
    }
    free(mm); free(cc); free(pp); free(fl);
    *n_drawn = last + 1;
    *n_over = over;
    return got;
}

/* Full amplitude matrix A[i][a] = lineshape(m_i; res r(a)) * Y_{y(a)}(theta_i, phi_i).
 * Computed in double, stored as double (dt=0) or rounded once to float (dt=1, C16). */
void pwa_gen_amplitudes(const double *m, const double *c, const double *p, int64_t N,
                        int n_res, const double *Mr, const double *Gr, int n,
                        const int32_t *res_of_wave, const int32_t *yid_of_wave, int dt, void *out)
{
#pragma omp parallel
    {
        double *bw = (double *)malloc(sizeof(double) * 2 * (size_t)n_res);
#pragma omp for schedule(static)
        for (int64_t i = 0; i < N; ++i) {
            double yr[4], yi[4];
            for (int k = 0; k < 4; ++k) ylm(k, c[i], p[i], &yr[k], &yi[k]);
            for (int r = 0; r < n_res; ++r) lineshape(m[i], Mr[r], Gr[r], &bw[2 * r], &bw[2 * r + 1]);
            for (int a = 0; a < n; ++a) {
                int r = res_of_wave[a], y = yid_of_wave[a];
                double ar = bw[2 * r] * yr[y] - bw[2 * r + 1] * yi[y];
                double ai = bw[2 * r] * yi[y] + bw[2 * r + 1] * yr[y];
                if (dt) { ((float *)out)[(i * n + a) * 2] = (float)ar; ((float *)out)[(i * n + a) * 2 + 1] = (float)ai; }
                else    { ((double *)out)[(i * n + a) * 2] = ar;       ((double *)out)[(i * n + a) * 2 + 1] = ai; }
            }
        }
        free(bw);
    }
}

/* Angular factors only: Z[i][s] = Y_{yids[s]}(theta_i, phi_i)  (factored upload, cfg 3) */
void pwa_gen_angular(const double *c, const double *p, int64_t N, int n_ang,
                     const int32_t *yids, int dt, void *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i)
        for (int s = 0; s < n_ang; ++s) {
            double re, im;
            ylm(yids[s], c[i], p[i], &re, &im);
            if (dt) { ((float *)out)[(i * n_ang + s) * 2] = (float)re; ((float *)out)[(i * n_ang + s) * 2 + 1] = (float)im; }
            else    { ((double *)out)[(i * n_ang + s) * 2] = re;       ((double *)out)[(i * n_ang + s) * 2 + 1] = im; }
        }
}
