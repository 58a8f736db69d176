// minimize.cpp — host quasi-Newton driver (P:55 fn. 3: "-ln L is fed to the minimizer";
// P:89 names Minuit/Fumili; reading C17: plain BFGS in the 2n Cartesian reals of V with a
// backtracking Armijo line search).  Everything here is host code that only calls the ABI.
#include <math.h>
#include <string.h>

#include <vector>

#include "../../include/pwa.h"

namespace {

struct Bfgs {
    int d = 0;
    std::vector<double> x, g, H, p, xt, gt;
    double f = 0.0, t = 1.0, slope = 0.0;
    int iter = 0;
    bool done = false, have = false;

    void init(int dim, const double *x0)
    {
        d = dim; x.assign(x0, x0 + d); g.assign(d, 0.0); p.assign(d, 0.0); xt.assign(d, 0.0); gt.assign(d, 0.0);
        H.assign((size_t)d * d, 0.0);
        for (int i = 0; i < d; ++i) H[(size_t)i * d + i] = 1.0;
    }
    double gmax() const { double m = 0.0; for (double v : g) m = fmax(m, fabs(v)); return m; }
    void direction(bool first)
    {
        for (int i = 0; i < d; ++i) { double s = 0.0; for (int j = 0; j < d; ++j) s -= H[(size_t)i * d + j] * g[j]; p[i] = s; }
        slope = 0.0; for (int i = 0; i < d; ++i) slope += p[i] * g[i];
        if (!(slope < 0.0)) {   // not a descent direction: reset
            for (size_t k = 0; k < H.size(); ++k) H[k] = 0.0;
            for (int i = 0; i < d; ++i) { H[(size_t)i * d + i] = 1.0; p[i] = -g[i]; }
            slope = 0.0; for (int i = 0; i < d; ++i) slope -= g[i] * g[i];
            first = true;
        }
        t = 1.0;
        if (first) { double nrm = 0.0; for (int i = 0; i < d; ++i) nrm += p[i] * p[i]; nrm = sqrt(nrm); if (nrm > 1.0) t = 1.0 / nrm; }
    }
    void trial() { for (int i = 0; i < d; ++i) xt[i] = x[i] + t * p[i]; }
    // returns true when the trial point was accepted
    bool update(double ft, int max_iter, double gtol)
    {
        const double c1 = 1e-4;
        if (!(isfinite(ft)) || ft > f + c1 * t * slope) {
            t *= 0.5;
            if (t < 1e-20) done = true;
            return false;
        }
        std::vector<double> s(d), y(d), Hy(d);
        double sy = 0.0;
        for (int i = 0; i < d; ++i) { s[i] = xt[i] - x[i]; y[i] = gt[i] - g[i]; sy += s[i] * y[i]; }
        x = xt; g = gt; f = ft; ++iter;
        double ss = 0.0, yy = 0.0;
        for (int i = 0; i < d; ++i) { ss += s[i] * s[i]; yy += y[i] * y[i]; }
        if (sy > 1e-12 * sqrt(ss * yy)) {
            if (iter == 1) { const double sc = sy / yy; for (int i = 0; i < d; ++i) H[(size_t)i * d + i] = sc; }
            double yHy = 0.0;
            for (int i = 0; i < d; ++i) { double v = 0.0; for (int j = 0; j < d; ++j) v += H[(size_t)i * d + j] * y[j]; Hy[i] = v; }
            for (int i = 0; i < d; ++i) yHy += y[i] * Hy[i];
            const double rho = 1.0 / sy;
            for (int i = 0; i < d; ++i)
                for (int j = 0; j < d; ++j)
                    H[(size_t)i * d + j] += -rho * (Hy[i] * s[j] + s[i] * Hy[j]) + (rho * rho * yHy + rho) * s[i] * s[j];
        }
        if (iter >= max_iter || gmax() < gtol) done = true;
        else direction(false);
        return true;
    }
};

}  // namespace

extern "C" {

pwa_status pwa_minimize_bfgs(pwa_ctx *ctx, double *V, int32_t max_iter, double gtol, double *nll_out,
                             int32_t *n_iter_out, int32_t *n_evals_out)
{
    int32_t evals = 0;
    pwa_status s = pwa_minimize_bfgs_batch(ctx, 1, V, max_iter, gtol, nll_out, &evals);
    if (n_evals_out) *n_evals_out = evals;
    if (n_iter_out) *n_iter_out = -1;
    return s;
}

// internal: dimension is discovered through a probe evaluation buffer sized by the caller's n
pwa_status pwa_minimize_bfgs_batch(pwa_ctx *ctx, int32_t K, double *V, int32_t max_iter, double gtol,
                                   double *nll_out, int32_t *n_evals_out)
{
    if (!ctx || !V || K < 1 || K > 1024 || max_iter < 0) return PWA_ERR_INVALID_ARG;
    const int n = pwa_n_waves(ctx), d = 2 * n;
    std::vector<Bfgs> fit(K);
    std::vector<double> X((size_t)K * d), F(K), Gr((size_t)K * d);
    memcpy(X.data(), V, sizeof(double) * (size_t)K * d);
    int32_t evals = 0;
    pwa_status worst = PWA_OK;
    auto eval = [&]() -> pwa_status {
        pwa_status s = (K == 1) ? pwa_nll_grad(ctx, X.data(), F.data(), Gr.data(), nullptr)
                                : pwa_nll_grad_batch(ctx, K, X.data(), F.data(), Gr.data(), nullptr);
        evals += 1;
        if (s == PWA_WARN_NONFINITE) { worst = s; return PWA_OK; }
        return s;
    };
    pwa_status s = eval();
    if (s != PWA_OK) return s;
    // the K fits are independent: their O(d^2) updates run on the host cores in parallel (the results do not
    // depend on the thread count: every fit is handled by exactly one thread)
#pragma omp parallel for schedule(static) if (K >= 4)
    for (int k = 0; k < K; ++k) {
        fit[k].init(d, X.data() + (size_t)k * d);
        fit[k].f = F[k];
        memcpy(fit[k].g.data(), Gr.data() + (size_t)k * d, sizeof(double) * d);
        if (max_iter == 0 || fit[k].gmax() < gtol) fit[k].done = true;
        else fit[k].direction(true);
    }
    for (;;) {
        bool any = false;
        for (int k = 0; k < K; ++k) {
            if (!fit[k].done) { fit[k].trial(); any = true; memcpy(X.data() + (size_t)k * d, fit[k].xt.data(), sizeof(double) * d); }
            else memcpy(X.data() + (size_t)k * d, fit[k].x.data(), sizeof(double) * d);
        }
        if (!any) break;
        s = eval();
        if (s != PWA_OK) return s;
#pragma omp parallel for schedule(static) if (K >= 4)
        for (int k = 0; k < K; ++k) {
            if (fit[k].done) continue;
            memcpy(fit[k].gt.data(), Gr.data() + (size_t)k * d, sizeof(double) * d);
            fit[k].update(F[k], max_iter, gtol);
        }
    }
    for (int k = 0; k < K; ++k) {
        memcpy(V + (size_t)k * d, fit[k].x.data(), sizeof(double) * d);
        if (nll_out) nll_out[k] = fit[k].f;
    }
    if (n_evals_out) *n_evals_out = evals;
    return worst;
}

}  // extern "C"
