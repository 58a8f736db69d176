/*
 * pwa_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct restatement of the extended log-likelihood of
 * arXiv 1108.5882 ("Partial Wave Analysis using Graphics Cards", N. Berger) and of its
 * gradient with respect to the complex production amplitudes V.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * this file.  It shares no code, header, table or helper with the CUDA library in
 * paper_1108_5882_b200/csrc/, and neither side includes or imports the other.
 *
 * Citations: "P:n" = /root/reference/PAPER.md line n.  "C<k>" = reading number k listed
 * in DESIGN.md section 3 (points on which the paper is silent).
 *
 *   eq. 1:  I(Omega) = | sum_a V_a A_a(Omega) |^2
 *   eq. 3:  ln L = sum_i ln( sum_a sum_a' V_a V_a'^* A_a(Om_i) A_a'^*(Om_i) )
 *                        - sum_a sum_a' V_a V_a'^* ( 1/N_gen sum_j A_a(Om_j) A_a'^*(Om_j) )
 *   P:55 fn. 3  :  -ln L is what the minimiser receives.
 *
 * Notation:  A[i][a] data amplitudes (N x n), B[j][a] accepted-MC
 * amplitudes (N_acc x n), S_i = sum_a V_a A_ia, L_data = sum_i ln|S_i|^2,
 * Norm(V) = (1/N_gen) sum_j |sum_a V_a B_ja|^2 = V^H M V with M = B^H B / N_gen (C1),
 * T_a = sum_i A_ia / S_i,  nll = -(L_data - Norm),
 * g_a = d nll/d Re V_a + i d nll/d Im V_a = -2 conj(T_a) + 2 (M V)_a   (C6).
 *
 * Arithmetic: every product and quotient in IEEE double; the per-event coherent sum over
 * waves runs in wave-index order in long double (>= fp64, so the oracle's own rounding is
 * below the GPU's); every sum over events is Neumaier-compensated ("the numerical
 * result is strongly dependent on the summing algorithm") with per-thread partials that
 * are combined in thread order.  No blocking, fusion or reordering beyond that.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): P1 single-wave closed form,
 * P2 global-phase invariance, P3 M Hermitian PSD, P4 V^H M V == explicit MC sum and the
 * transposed pairing fails, P5 gradient vs central differences, P6 eq.1 == eq.3 double
 * sum on dyadic inputs, P7 Euler identity sum_a V_a T_a = N, P8 numpy BLAS (zgemm/zgemv),
 * P9 permutation / duplication / scaling invariances, P10 Breit-Wigner closed forms and
 * derivative vs differences, brute-force pure-Python on tiny inputs; P13 eq. 2 form: scale
 * invariance, finite differences, equality with eq. 3 at Norm = N_data; P14 polar chain rule vs
 * finite differences in (r, phi); P15 Fumili matrix: H_data V = 2 grad(L_data) (Euler), numpy
 * restatement, PSD, Hess(Norm) vs differences of the norm gradient; P16 event weights: unit weights,
 * integer weights = duplicated events, numpy restatement, linearity in w; P17 the sampled entry points
 * (norm_block / norm_block_w with a0, b0 > 0, fumili_rows with p0 > 0): bitwise equal to the same entries of
 * the full result, zero outside, numpy restatement of the block; P18 fixed-phase gauge: nll unchanged, the turned
 * gradient equals the gradient evaluated at the turned V, relative phases kept, gauge identity sum_a (x g_y - y g_x) = 0.
 * Parity unpinned by the paper: the choices C2, C3, C4, C5, C9-C13 (definitions, not
 * results), and the resonance-parameter gradient beyond finite differences (P5/P10 style).
 *
 * Storage flag `dt`: 0 = amplitudes stored as double (re,im interleaved), 1 = stored as
 * float (re,im interleaved) and widened on load (exact) — C16.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---------- Neumaier compensated accumulator ---------------------------------------- */
typedef struct { double s, c; } nsum;

static inline void nadd(nsum *a, double x)
{
    double t = a->s + x;
    if (!isfinite(t)) { a->s = t; return; }   /* C14: +-inf / nan propagate as plain IEEE sums */
    if (fabs(a->s) >= fabs(x)) a->c += (a->s - t) + x;
    else                       a->c += (x - t) + a->s;
    a->s = t;
}
static inline double nval(const nsum *a) { return a->s + a->c; }
static inline void nmerge(nsum *dst, const nsum *src) { nadd(dst, src->s); nadd(dst, src->c); }

static inline double ld_amp(const void *p, int dt, int64_t idx)
{
    return dt ? (double)((const float *)p)[idx] : ((const double *)p)[idx];
}

static int n_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
int pwa_oracle_threads(void) { return n_threads(); }
void pwa_oracle_set_threads(int t)
{
#ifdef _OPENMP
    if (t > 0) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

/* ---------- Breit-Wigner (C3): BW(m; M, G) = 1 / (M^2 - m^2 - i M G) ----------------- */
void pwa_oracle_bw(double m, double M, double G, double out[2])
{
    double dre = M * M - m * m;     /* denominator d = dre + i*dim */
    double dim = -M * G;
    double den = dre * dre + dim * dim;
    out[0] = dre / den;             /* 1/d = conj(d)/|d|^2 */
    out[1] = -dim / den;
}

/* dBW/dM = -(2M - iG) BW^2 ;  dBW/dG = i M BW^2   (differentiate 1/d, d = M^2-m^2-iMG) */
void pwa_oracle_bw_deriv(double m, double M, double G, double dM[2], double dG[2])
{
    double bw[2], sq[2];
    pwa_oracle_bw(m, M, G, bw);
    sq[0] = bw[0] * bw[0] - bw[1] * bw[1];
    sq[1] = 2.0 * bw[0] * bw[1];
    /* -(2M - iG) * sq */
    dM[0] = -(2.0 * M * sq[0] + G * sq[1]);
    dM[1] = -(2.0 * M * sq[1] - G * sq[0]);
    /* i M * sq */
    dG[0] = -M * sq[1];
    dG[1] = M * sq[0];
}

/* ---------- factored mode, step 1: A_ia = BW(m_i; M_r(a), G_r(a)) * Z_{i,s(a)} -- */
void pwa_oracle_expand_factored(const double *mass, const void *Z, int dtZ, int n_ang,
                                int64_t N, int n, const int32_t *res_of_wave,
                                const int32_t *ang_of_wave, const double *Mr,
                                const double *Gr, double *A_out)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < N; ++i) {
        for (int a = 0; a < n; ++a) {
            double bw[2];
            int r = res_of_wave[a], s = ang_of_wave[a];
            pwa_oracle_bw(mass[i], Mr[r], Gr[r], bw);
            double zr = ld_amp(Z, dtZ, (i * n_ang + s) * 2);
            double zi = ld_amp(Z, dtZ, (i * n_ang + s) * 2 + 1);
            A_out[(i * n + a) * 2]     = bw[0] * zr - bw[1] * zi;
            A_out[(i * n + a) * 2 + 1] = bw[0] * zi + bw[1] * zr;
        }
    }
}

/* ---------- data term: steps 2-5 ------------------------------------------------------
 * S_i = sum_a V_a A_ia (eq. 1);  l_i = ln|S_i|^2 (eq. 3 first term);
 * L = sum_i l_i;  T_a = sum_i A_ia / S_i.   Returns the number of events with I_i == 0
 * or non-finite l_i (C14: IEEE values propagate). */
/* NEXT-3: optional per-event weights w_i (NULL = all 1):
 * L = sum_i w_i l_i, T_a = sum_i w_i A_ia / S_i (a weighted unbinned likelihood; weights that are
 * small non-negative integers are exactly event multiplicities). */
int64_t pwa_oracle_data_term_w(const void *A, int dt, int64_t N, int n, const double *V, const double *w,
                               double *L_out, double *T_out /* [n][2] */)
{
    int nt = n_threads();
    nsum *part = (nsum *)calloc((size_t)nt * (size_t)(1 + 2 * n), sizeof(nsum));
    int64_t bad = 0;
#pragma omp parallel num_threads(nt) reduction(+ : bad)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        nsum *my = part + (size_t)tid * (size_t)(1 + 2 * n);
#pragma omp for schedule(static)
        for (int64_t i = 0; i < N; ++i) {
            long double sr = 0.0L, si = 0.0L;
            for (int a = 0; a < n; ++a) {
                double ar = ld_amp(A, dt, (i * n + a) * 2);
                double ai = ld_amp(A, dt, (i * n + a) * 2 + 1);
                sr += (long double)V[2 * a] * ar - (long double)V[2 * a + 1] * ai;
                si += (long double)V[2 * a] * ai + (long double)V[2 * a + 1] * ar;
            }
            double Sr = (double)sr, Si = (double)si;
            double I = Sr * Sr + Si * Si;
            double l = log(I);
            const double wi = w ? w[i] : 1.0;
            if (!(I > 0.0) || !isfinite(l)) bad += 1;
            nadd(&my[0], wi * l);
            for (int a = 0; a < n; ++a) {
                double ar = ld_amp(A, dt, (i * n + a) * 2);
                double ai = ld_amp(A, dt, (i * n + a) * 2 + 1);
                /* A / S = A * conj(S) / I */
                nadd(&my[1 + 2 * a], wi * ((ar * Sr + ai * Si) / I));
                nadd(&my[2 + 2 * a], wi * ((ai * Sr - ar * Si) / I));
            }
        }
    }
    for (int k = 0; k < 1 + 2 * n; ++k) {
        nsum tot = {0.0, 0.0};
        for (int t = 0; t < nt; ++t) nmerge(&tot, &part[(size_t)t * (size_t)(1 + 2 * n) + k]);
        if (k == 0) *L_out = nval(&tot);
        else        T_out[k - 1] = nval(&tot);
    }
    free(part);
    return bad;
}

int64_t pwa_oracle_data_term(const void *A, int dt, int64_t N, int n, const double *V,
                             double *L_out, double *T_out /* [n][2] */)
{
    return pwa_oracle_data_term_w(A, dt, N, n, V, NULL, L_out, T_out);
}

/* ---------- normalisation matrix: step 6 (P:41 inner bracket, C1) ---------------------
 * M_ab = (1/N_gen) sum_j conj(B_ja) B_jb  for ALL (a,b): Hermitian symmetry is NOT used
 * here so that it can be tested. Only entries with a in [a0,a1) and b in [b0,b1) are
 * computed (others left untouched) so single entries can be sampled at full size. */
/* Optional per-event MC weights w_j (NULL = all 1), P:37 fn. 2 ("it is also possible to generate
 * events unevenly ... and then weight them"): M_ab = (1/N_gen) sum_j w_j conj(B_ja) B_jb. */
void pwa_oracle_norm_block_w(const void *B, int dt, int64_t N_acc, int n, int64_t N_gen, const double *w,
                             int a0, int a1, int b0, int b1, double *M_out /* [n][n][2] */)
{
    int nt = n_threads();
    int na = a1 - a0, nb = b1 - b0;
    size_t per = (size_t)na * (size_t)nb * 2;
    nsum *part = (nsum *)calloc((size_t)nt * per, sizeof(nsum));
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        nsum *my = part + (size_t)tid * per;
#pragma omp for schedule(static)
        for (int64_t j = 0; j < N_acc; ++j) {
            const double wj = w ? w[j] : 1.0;
            for (int a = a0; a < a1; ++a) {
                double ar = ld_amp(B, dt, (j * n + a) * 2);
                double ai = ld_amp(B, dt, (j * n + a) * 2 + 1);
                for (int b = b0; b < b1; ++b) {
                    double br = ld_amp(B, dt, (j * n + b) * 2);
                    double bi = ld_amp(B, dt, (j * n + b) * 2 + 1);
                    size_t k = ((size_t)(a - a0) * (size_t)nb + (size_t)(b - b0)) * 2;
                    /* conj(a) * b = (ar - i ai)(br + i bi) */
                    nadd(&my[k],     wj * (ar * br + ai * bi));
                    nadd(&my[k + 1], wj * (ar * bi - ai * br));
                }
            }
        }
    }
    for (int a = a0; a < a1; ++a)
        for (int b = b0; b < b1; ++b)
            for (int c = 0; c < 2; ++c) {
                size_t k = ((size_t)(a - a0) * (size_t)nb + (size_t)(b - b0)) * 2 + (size_t)c;
                nsum tot = {0.0, 0.0};
                for (int t = 0; t < nt; ++t) nmerge(&tot, &part[(size_t)t * per + k]);
                M_out[((size_t)a * (size_t)n + (size_t)b) * 2 + (size_t)c] = nval(&tot) / (double)N_gen;
            }
    free(part);
}

void pwa_oracle_norm_block(const void *B, int dt, int64_t N_acc, int n, int64_t N_gen,
                           int a0, int a1, int b0, int b1, double *M_out /* [n][n][2] */)
{
    pwa_oracle_norm_block_w(B, dt, N_acc, n, N_gen, NULL, a0, a1, b0, b1, M_out);
}

void pwa_oracle_norm_matrix(const void *B, int dt, int64_t N_acc, int n, int64_t N_gen,
                            double *M_out)
{
    pwa_oracle_norm_block(B, dt, N_acc, n, N_gen, 0, n, 0, n, M_out);
}

/* ---------- explicit MC sum: step 7 second form (P:41 second term via eq. 1) ----------
 * Norm' = (1/N_gen) sum_j |sum_a V_a B_ja|^2 ;  gN'_a = (2/N_gen) sum_j conj(B_ja) S_j  */
void pwa_oracle_norm_explicit(const void *B, int dt, int64_t N_acc, int n, int64_t N_gen,
                              const double *V, double *Norm_out, double *gN_out /* [n][2] or NULL */)
{
    int nt = n_threads();
    size_t per = (size_t)(1 + 2 * n);
    nsum *part = (nsum *)calloc((size_t)nt * per, sizeof(nsum));
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        nsum *my = part + (size_t)tid * per;
#pragma omp for schedule(static)
        for (int64_t j = 0; j < N_acc; ++j) {
            long double sr = 0.0L, si = 0.0L;
            for (int a = 0; a < n; ++a) {
                double br = ld_amp(B, dt, (j * n + a) * 2);
                double bi = ld_amp(B, dt, (j * n + a) * 2 + 1);
                sr += (long double)V[2 * a] * br - (long double)V[2 * a + 1] * bi;
                si += (long double)V[2 * a] * bi + (long double)V[2 * a + 1] * br;
            }
            double Sr = (double)sr, Si = (double)si;
            nadd(&my[0], Sr * Sr + Si * Si);
            for (int a = 0; a < n; ++a) {
                double br = ld_amp(B, dt, (j * n + a) * 2);
                double bi = ld_amp(B, dt, (j * n + a) * 2 + 1);
                nadd(&my[1 + 2 * a], br * Sr + bi * Si);   /* Re conj(B) S */
                nadd(&my[2 + 2 * a], br * Si - bi * Sr);   /* Im conj(B) S */
            }
        }
    }
    for (size_t k = 0; k < per; ++k) {
        nsum tot = {0.0, 0.0};
        for (int t = 0; t < nt; ++t) nmerge(&tot, &part[(size_t)t * per + k]);
        if (k == 0) *Norm_out = nval(&tot) / (double)N_gen;
        else if (gN_out) gN_out[k - 1] = 2.0 * nval(&tot) / (double)N_gen;
    }
    free(part);
}

/* ---------- steps 7-8: Norm = V^H M V ; nll = -(L - Norm) ; g = -2 conj(T) + 2 M V ---- */
void pwa_oracle_assemble(int n, double L, const double *T, const double *M, const double *V,
                         double *nll, double *grad /* [n][2] */, double *parts /* [2] or NULL */)
{
    nsum nrm = {0.0, 0.0};
    for (int a = 0; a < n; ++a) {
        nsum mr = {0.0, 0.0}, mi = {0.0, 0.0};     /* (M V)_a */
        for (int b = 0; b < n; ++b) {
            double Mr = M[(a * n + b) * 2], Mi = M[(a * n + b) * 2 + 1];
            nadd(&mr, Mr * V[2 * b]);  nadd(&mr, -Mi * V[2 * b + 1]);
            nadd(&mi, Mr * V[2 * b + 1]);  nadd(&mi, Mi * V[2 * b]);
        }
        double mvr = nval(&mr), mvi = nval(&mi);
        /* Re( conj(V_a) (MV)_a ) ; the imaginary parts cancel in the Hermitian form */
        nadd(&nrm, V[2 * a] * mvr);  nadd(&nrm, V[2 * a + 1] * mvi);
        grad[2 * a]     = -2.0 * T[2 * a] + 2.0 * mvr;         /* -2 Re conj(T) = -2 Re T */
        grad[2 * a + 1] =  2.0 * T[2 * a + 1] + 2.0 * mvi;     /* -2 Im conj(T) = +2 Im T */
    }
    double Nv = nval(&nrm);
    *nll = -(L - Nv);
    if (parts) { parts[0] = L; parts[1] = Nv; }
}

/* ---------- NEXT-4 variants: eq. 2 form and polar parameters ------------
 * eq. 2: L = prod_i I(Om_i) / integral(eps I).  With the integral done as the MC sum of
 * eq. 3, integral = Norm(V) = V^H M V, so
 *     ln L2 = L_data - N_data ln Norm,   nll2 = -L_data + N_data ln Norm,
 *     g(nll2) = -2 conj(T) + (2 N_data / Norm) M V.
 * Invariant under V -> s V (the overall scale is not a parameter of eq. 2).                       */
void pwa_oracle_assemble_eq2(int n, double N_data, double L, const double *T, const double *M,
                             const double *V, double *nll, double *grad, double *parts)
{
    double nll3, p3[2];
    double *g3 = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    double *zero = (double *)calloc(2 * (size_t)n, sizeof(double));
    pwa_oracle_assemble(n, 0.0, zero, M, V, &nll3, g3, p3);      /* g3 = 2 M V, p3[1] = Norm */
    double Nv = p3[1];
    *nll = -L + N_data * log(Nv);
    for (int a = 0; a < n; ++a) {
        grad[2 * a]     = -2.0 * T[2 * a]     + (N_data / Nv) * g3[2 * a];
        grad[2 * a + 1] =  2.0 * T[2 * a + 1] + (N_data / Nv) * g3[2 * a + 1];
    }
    if (parts) { parts[0] = L; parts[1] = Nv; }
    free(g3); free(zero);
}

/* Polar parameters: V_a = r_a exp(i phi_a).  Chain rule on a Cartesian gradient
 * (gx, gy) = (d f/d Re V_a, d f/d Im V_a):  d f/d r = gx cos(phi) + gy sin(phi),
 * d f/d phi = -gx r sin(phi) + gy r cos(phi) = -Im V gx + Re V gy.  out: [n][2] = (d/dr, d/dphi). */
void pwa_oracle_grad_polar(int n, const double *V, const double *grad, double *out)
{
    for (int a = 0; a < n; ++a) {
        double x = V[2 * a], y = V[2 * a + 1], r = hypot(x, y), phi = atan2(y, x);
        out[2 * a]     = grad[2 * a] * cos(phi) + grad[2 * a + 1] * sin(phi);
        out[2 * a + 1] = -grad[2 * a] * r * sin(phi) + grad[2 * a + 1] * r * cos(phi);
    }
}

/* Fixed-phase gauge.  |S_i| and V^dagger M V do not change under V -> exp(i a) V, so nll
 * (eq. 3 and eq. 2) has one flat direction.  The gauge "wave ref is real and non-negative" removes it: with
 * a = -arg V_ref every V_a is turned by a; a Cartesian gradient, read as the complex number g_a = d/dx_a + i d/dy_a,
 * turns by the same angle (nll(V) = nll(V') with V' = exp(i a) V gives g'(V') = exp(i a) g(V)); the component
 * d/d Im V_ref belongs to the parameter the gauge fixes at zero and is dropped (set to 0).  In place; grad may be NULL. */
void pwa_oracle_fix_phase(int n, int ref, double *V, double *grad)
{
    double a = -atan2(V[2 * ref + 1], V[2 * ref]);
    for (int w = 0; w < n; ++w) {
        double r = hypot(V[2 * w], V[2 * w + 1]), ph = atan2(V[2 * w + 1], V[2 * w]);
        V[2 * w] = r * cos(ph + a);
        V[2 * w + 1] = r * sin(ph + a);
        if (grad) {
            double gr = hypot(grad[2 * w], grad[2 * w + 1]), gp = atan2(grad[2 * w + 1], grad[2 * w]);
            grad[2 * w] = gr * cos(gp + a);
            grad[2 * w + 1] = gr * sin(gp + a);
        }
    }
    V[2 * ref + 1] = 0.0;                     /* exactly on the gauge (sin of a rounded angle leaves ~1e-17 r) */
    if (grad) grad[2 * ref + 1] = 0.0;
}

/* ---------- NEXT-2: Fumili-style approximate Hessian (ref. P:123) -----
 * For l_i = ln I_i the exact second derivative is (d2 I)/I - (dI)(dI)^T / I^2; Fumili keeps the
 * outer-product term only.  With u_i = d l_i / d(x_0, y_0, x_1, ...) = (2 Re t_i0, -2 Im t_i0, ...),
 * t_ia = A_ia / S_i:
 *     H_data = sum_i u_i u_i^T          (2n x 2n, symmetric, positive semi-definite)
 *     H      = H_data + Hess(Norm),  Hess(Norm) = 2 [[Re M_ab, -Im M_ab], [Im M_ab, Re M_ab]]  (exact: Norm is quadratic)
 * approximates the Hessian of nll = -(L_data - Norm).  H: [2n][2n] row-major; M may be NULL (H_data only). */
/* rows p0 <= p < p1 of H_data only (others untouched): per-thread compensated partials over events,
 * merged in thread order, as in the data term.  For sampled checks at full size. */
void pwa_oracle_fumili_rows(const void *A, int dt, int64_t N, int n, const double *V, int p0, int p1, double *H)
{
    const int D = 2 * n, nr = p1 - p0;
    int nt = n_threads();
    size_t per = (size_t)nr * D;
    nsum *part = (nsum *)calloc((size_t)nt * per, sizeof(nsum));
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        nsum *my = part + (size_t)tid * per;
        double *u = (double *)malloc(sizeof(double) * D);
#pragma omp for schedule(static)
        for (int64_t i = 0; i < N; ++i) {
            long double sr = 0.0L, si = 0.0L;
            for (int a = 0; a < n; ++a) {
                double ar = ld_amp(A, dt, (i * n + a) * 2), ai = ld_amp(A, dt, (i * n + a) * 2 + 1);
                sr += (long double)V[2 * a] * ar - (long double)V[2 * a + 1] * ai;
                si += (long double)V[2 * a] * ai + (long double)V[2 * a + 1] * ar;
            }
            double Sr = (double)sr, Si = (double)si, I = Sr * Sr + Si * Si;
            for (int a = 0; a < n; ++a) {
                double ar = ld_amp(A, dt, (i * n + a) * 2), ai = ld_amp(A, dt, (i * n + a) * 2 + 1);
                /* t = A / S = A conj(S) / I */
                double tr = (ar * Sr + ai * Si) / I, ti = (ai * Sr - ar * Si) / I;
                u[2 * a] = 2.0 * tr;  u[2 * a + 1] = -2.0 * ti;
            }
            for (int p = p0; p < p1; ++p)
                for (int q = 0; q < D; ++q) nadd(&my[(size_t)(p - p0) * D + q], u[p] * u[q]);
        }
        free(u);
    }
    for (size_t k = 0; k < per; ++k) {
        nsum tot = {0.0, 0.0};
        for (int t = 0; t < nt; ++t) nmerge(&tot, &part[(size_t)t * per + k]);
        H[(size_t)p0 * D + k] = nval(&tot);
    }
    free(part);
}

void pwa_oracle_fumili(const void *A, int dt, int64_t N, int n, const double *V, const double *M, double *H)
{
    const int D = 2 * n;
    pwa_oracle_fumili_rows(A, dt, N, n, V, 0, D, H);
    if (M)
        for (int a = 0; a < n; ++a)
            for (int b = 0; b < n; ++b) {
                double Mr = M[(a * n + b) * 2], Mi = M[(a * n + b) * 2 + 1];
                H[(2 * a) * D + 2 * b] += 2.0 * Mr;          H[(2 * a) * D + 2 * b + 1] += -2.0 * Mi;
                H[(2 * a + 1) * D + 2 * b] += 2.0 * Mi;      H[(2 * a + 1) * D + 2 * b + 1] += 2.0 * Mr;
            }
}

int64_t pwa_oracle_nll_grad(const void *A, int dt, int64_t N, int n, const double *M,
                            const double *V, double *nll, double *grad, double *parts)
{
    double L;
    double *T = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    int64_t bad = pwa_oracle_data_term(A, dt, N, n, V, &L, T);
    pwa_oracle_assemble(n, L, T, M, V, nll, grad, parts);
    free(T);
    return bad;
}

/* step 9: batched = loop over k, no cleverness. V: [K][n][2]. */
int64_t pwa_oracle_nll_grad_batch(const void *A, int dt, int64_t N, int n, const double *M,
                                  int K, const double *V, double *nll, double *grad, double *parts)
{
    int64_t bad = 0;
    for (int k = 0; k < K; ++k)
        bad += pwa_oracle_nll_grad(A, dt, N, n, M, V + (size_t)k * 2 * (size_t)n, nll + k,
                                   grad + (size_t)k * 2 * (size_t)n, parts ? parts + 2 * k : NULL);
    return bad;
}

/* step 10: eq. 3 literally for ONE event (the paper's n^2 lookup form):
 * I' = sum_a sum_a' V_a conj(V_a') A_a conj(A_a').  Returns (Re I', Im I'). */
void pwa_oracle_intensity_eq3(const double *Arow, int n, const double *V, double out[2])
{
    double re = 0.0, im = 0.0;
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b) {
            /* V_a conj(V_b) */
            double vr = V[2 * a] * V[2 * b] + V[2 * a + 1] * V[2 * b + 1];
            double vi = V[2 * a + 1] * V[2 * b] - V[2 * a] * V[2 * b + 1];
            /* A_a conj(A_b) */
            double ar = Arow[2 * a] * Arow[2 * b] + Arow[2 * a + 1] * Arow[2 * b + 1];
            double ai = Arow[2 * a + 1] * Arow[2 * b] - Arow[2 * a] * Arow[2 * b + 1];
            re += vr * ar - vi * ai;
            im += vr * ai + vi * ar;
        }
    out[0] = re; out[1] = im;
}

/* eq. 1 for ONE event: I = |sum_a V_a A_a|^2 */
double pwa_oracle_intensity_eq1(const double *Arow, int n, const double *V)
{
    double sr = 0.0, si = 0.0;
    for (int a = 0; a < n; ++a) {
        sr += V[2 * a] * Arow[2 * a] - V[2 * a + 1] * Arow[2 * a + 1];
        si += V[2 * a] * Arow[2 * a + 1] + V[2 * a + 1] * Arow[2 * a];
    }
    return sr * sr + si * si;
}

/* ---------- gradient w.r.t. floating resonance parameters (reading A9) ----------------
 * For one sample X (data or MC) in factored form and resonance r:
 *   d_theta S_i = ( sum_{a: r(a)=r} V_a Z_{i,s(a)} ) * d_theta BW(m_i; M_r, G_r)
 *   mode 0 (data): out_theta = 2 sum_i Re( d_theta S_i / S_i )           = d L_data / d theta
 *   mode 1 (MC)  : out_theta = (2/N_gen) sum_j Re( conj(S_j) d_theta S_j ) = d Norm / d theta
 * dM_out, dG_out: [n_res].  N_gen ignored in mode 0. */
void pwa_oracle_res_grad(const double *mass, const void *Z, int dtZ, int n_ang, int64_t N,
                         int n, int n_res, const int32_t *res_of_wave,
                         const int32_t *ang_of_wave, const double *Mr, const double *Gr,
                         const double *V, int mode, int64_t N_gen, double *dM_out, double *dG_out)
{
    int nt = n_threads();
    size_t per = (size_t)(2 * n_res);
    nsum *part = (nsum *)calloc((size_t)nt * per, sizeof(nsum));
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
        int tid = omp_get_thread_num();
#else
        int tid = 0;
#endif
        nsum *my = part + (size_t)tid * per;
#pragma omp for schedule(static)
        for (int64_t i = 0; i < N; ++i) {
            long double sr = 0.0L, si = 0.0L;
            for (int a = 0; a < n; ++a) {
                double bw[2];
                int r = res_of_wave[a], s = ang_of_wave[a];
                pwa_oracle_bw(mass[i], Mr[r], Gr[r], bw);
                double zr = ld_amp(Z, dtZ, (i * n_ang + s) * 2);
                double zi = ld_amp(Z, dtZ, (i * n_ang + s) * 2 + 1);
                double ar = bw[0] * zr - bw[1] * zi, ai = bw[0] * zi + bw[1] * zr;
                sr += (long double)V[2 * a] * ar - (long double)V[2 * a + 1] * ai;
                si += (long double)V[2 * a] * ai + (long double)V[2 * a + 1] * ar;
            }
            double Sr = (double)sr, Si = (double)si, I = Sr * Sr + Si * Si;
            for (int r = 0; r < n_res; ++r) {
                double wr = 0.0, wi = 0.0;   /* w = sum_{a: r(a)=r} V_a Z_{i,s(a)} */
                for (int a = 0; a < n; ++a) {
                    if (res_of_wave[a] != r) continue;
                    int s = ang_of_wave[a];
                    double zr = ld_amp(Z, dtZ, (i * n_ang + s) * 2);
                    double zi = ld_amp(Z, dtZ, (i * n_ang + s) * 2 + 1);
                    wr += V[2 * a] * zr - V[2 * a + 1] * zi;
                    wi += V[2 * a] * zi + V[2 * a + 1] * zr;
                }
                double dM[2], dG[2];
                pwa_oracle_bw_deriv(mass[i], Mr[r], Gr[r], dM, dG);
                double dSM_r = wr * dM[0] - wi * dM[1], dSM_i = wr * dM[1] + wi * dM[0];
                double dSG_r = wr * dG[0] - wi * dG[1], dSG_i = wr * dG[1] + wi * dG[0];
                if (mode == 0) {   /* Re(dS / S) = Re(dS conj(S)) / I */
                    nadd(&my[2 * r],     2.0 * (dSM_r * Sr + dSM_i * Si) / I);
                    nadd(&my[2 * r + 1], 2.0 * (dSG_r * Sr + dSG_i * Si) / I);
                } else {           /* Re(conj(S) dS) */
                    nadd(&my[2 * r],     2.0 * (dSM_r * Sr + dSM_i * Si));
                    nadd(&my[2 * r + 1], 2.0 * (dSG_r * Sr + dSG_i * Si));
                }
            }
        }
    }
    for (int r = 0; r < n_res; ++r)
        for (int c = 0; c < 2; ++c) {
            nsum tot = {0.0, 0.0};
            for (int t = 0; t < nt; ++t) nmerge(&tot, &part[(size_t)t * per + (size_t)(2 * r + c)]);
            double v = nval(&tot);
            if (mode == 1) v /= (double)N_gen;
            if (c == 0) dM_out[r] = v; else dG_out[r] = v;
        }
    free(part);
}
