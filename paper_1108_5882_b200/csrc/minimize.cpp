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
    std::vector<double> cap;  // optional: largest |step| per variable and iteration (0 = unlimited); keeps a resonance in its basin
    double f = 0.0, t = 1.0, slope = 0.0;
    int iter = 0;
    int small_steps = 0;      // consecutive accepted steps shorter than 2^-10 of the quasi-Newton step
    int stall_limit = 0;      // > 0: that many of them in a row end the fit with PWA_FIT_LINE_SEARCH (noisy evaluations, see batch_ex)
    bool fresh = true;        // the current direction is steepest descent (H = identity): a failed search along it is final
    int why = 0;              // why the fit stopped: PWA_FIT_CONVERGED / PWA_FIT_MAX_ITER / PWA_FIT_LINE_SEARCH
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
        fresh = first;
        t = 1.0;
        if (first) { double nrm = 0.0; for (int i = 0; i < d; ++i) nrm += p[i] * p[i]; nrm = sqrt(nrm); if (nrm > 1.0) t = 1.0 / nrm; }
        if (!cap.empty())
            for (int i = 0; i < d; ++i) if (cap[i] > 0.0 && fabs(p[i]) * t > cap[i]) t = cap[i] / fabs(p[i]);
    }
    void trial() { for (int i = 0; i < d; ++i) xt[i] = x[i] + t * p[i]; }
    // returns true when the trial point was accepted
    bool update(double ft, int max_iter, double gtol)
    {
        const double c1 = 1e-4;
        if (!(isfinite(ft)) || ft > f + c1 * t * slope) {
            t *= 0.5;
            if (t < 1e-20) {
                // the search along the quasi-Newton direction is exhausted: an inverse Hessian that has gone bad looks the
                // same as the resolution of nll, so restart once from steepest descent before giving up
                if (!fresh) {
                    for (size_t k = 0; k < H.size(); ++k) H[k] = 0.0;
                    for (int i = 0; i < d; ++i) H[(size_t)i * d + i] = 1.0;
                    direction(true);
                } else { done = true; why = PWA_FIT_LINE_SEARCH; }
            }
            return false;
        }
        std::vector<double> s(d), y(d), Hy(d);
        double sy = 0.0;
        for (int i = 0; i < d; ++i) { s[i] = xt[i] - x[i]; y[i] = gt[i] - g[i]; sy += s[i] * y[i]; }
        x = xt; g = gt; f = ft; ++iter;
        small_steps = (t < 0x1p-10 && iter > 1) ? small_steps + 1 : 0;
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
        if (gmax() < gtol) { done = true; why = PWA_FIT_CONVERGED; }
        else if (iter >= max_iter) { done = true; why = PWA_FIT_MAX_ITER; }
        else if (stall_limit > 0 && small_steps >= stall_limit) { done = true; why = PWA_FIT_LINE_SEARCH; }
        else direction(false);
        return true;
    }
};

}  // namespace

extern "C" {

pwa_status pwa_minimize_bfgs(pwa_ctx *ctx, double *V, int32_t max_iter, double gtol, double *nll_out,
                             int32_t *n_iter_out, int32_t *n_evals_out)
{
    return pwa_minimize_bfgs_batch_ex(ctx, 1, V, max_iter, gtol, nll_out, n_iter_out, nullptr, n_evals_out);
}

pwa_status pwa_minimize_bfgs_batch(pwa_ctx *ctx, int32_t K, double *V, int32_t max_iter, double gtol,
                                   double *nll_out, int32_t *n_evals_out)
{
    return pwa_minimize_bfgs_batch_ex(ctx, K, V, max_iter, gtol, nll_out, nullptr, nullptr, n_evals_out);
}

pwa_status pwa_minimize_bfgs_batch_ex(pwa_ctx *ctx, int32_t K, double *V, int32_t max_iter, double gtol,
                                      double *nll_out, int32_t *n_iter_out, int32_t *why_out, int32_t *n_evals_out)
{
    if (!ctx || !V || K < 1 || K > 1024 || max_iter < 0) return PWA_ERR_INVALID_ARG;
    const int n = pwa_n_waves(ctx), d = 2 * n;
    std::vector<Bfgs> fit(K);
    std::vector<double> X((size_t)K * d), F(K), Gr((size_t)K * d), Pt((size_t)K * 2);
    std::vector<int> act(K);                    // the fits evaluated by the current batched calls (all K in the first stage)
    for (int k = 0; k < K; ++k) act[k] = k;
    memcpy(X.data(), V, sizeof(double) * (size_t)K * d);
    // fixed-phase gauge ("fix_phase" = ref + 1): every starting point is turned so that Im V_ref = 0, and the
    // component d/dIm V_ref of every gradient is dropped.  BFGS then never moves that coordinate (its row of the inverse
    // Hessian stays the identity row, because the step and the gradient difference are zero there).
    int32_t gauge = 0;
    if (pwa_get_option(ctx, "fix_phase", &gauge) != PWA_OK) gauge = 0;
    const int ref = gauge - 1;
    if (ref >= 0) for (int k = 0; k < K; ++k) pwa_fix_phase_host(n, ref, X.data() + (size_t)k * d, nullptr);
    int32_t evals = 0;
    pwa_status worst = PWA_OK;
    auto eval = [&]() -> pwa_status {            // evaluates rows 0 .. act.size()-1 of X
        const int Ka = (int)act.size();
        pwa_status s = (Ka == 1) ? pwa_nll_grad(ctx, X.data(), F.data(), Gr.data(), Pt.data())
                                 : pwa_nll_grad_batch(ctx, Ka, X.data(), F.data(), Gr.data(), Pt.data());
        if (ref >= 0) for (int j = 0; j < Ka; ++j) Gr[(size_t)j * d + 2 * ref + 1] = 0.0;
        evals += 1;
        if (s == PWA_WARN_NONFINITE) { worst = s; return PWA_OK; }
        return s;
    };
    pwa_status s = eval();
    if (s != PWA_OK) return s;
    // Euler prescale (pin P7): along V -> s V the extended likelihood of eq. 3 is L_data + N ln s^2 - s^2 Norm, whose
    // optimum s^2 = N_data / Norm is known in closed form (at any stationary point Norm = N_data).  Starting there
    // removes the one direction in which a random start is wrong by orders of magnitude.  (eq. 2 is scale-invariant.)
    {
        int32_t lik = 0;
        const double n_data = (double)pwa_n_events(ctx, PWA_DATA);
        if (pwa_get_option(ctx, "likelihood", &lik) == PWA_OK && lik == 0 && n_data > 0.0 && max_iter > 0) {
            bool any = false;
            for (int k = 0; k < K; ++k) {
                const double norm = Pt[2 * k + 1];
                if (norm > 0.0 && isfinite(norm)) { const double sc = sqrt(n_data / norm); for (int i = 0; i < d; ++i) X[(size_t)k * d + i] *= sc; any = true; }
            }
            if (any) { s = eval(); if (s != PWA_OK) return s; }
        }
    }
    // the K fits are independent: their O(d^2) updates run on the host cores in parallel (the results do not
    // depend on the thread count: every fit is handled by exactly one thread)
#pragma omp parallel for schedule(static) if (K >= 4)
    for (int k = 0; k < K; ++k) {
        fit[k].init(d, X.data() + (size_t)k * d);
        fit[k].f = F[k];
        memcpy(fit[k].g.data(), Gr.data() + (size_t)k * d, sizeof(double) * d);
        if (fit[k].gmax() < gtol) { fit[k].done = true; fit[k].why = PWA_FIT_CONVERGED; }
        else if (max_iter == 0) { fit[k].done = true; fit[k].why = PWA_FIT_MAX_ITER; }
        else fit[k].direction(true);
    }
    auto lockstep = [&]() -> pwa_status {
        const int Ka = (int)act.size();
        for (;;) {
            bool any = false;
            for (int j = 0; j < Ka; ++j) {
                Bfgs &b = fit[act[j]];
                if (!b.done) { b.trial(); any = true; memcpy(X.data() + (size_t)j * d, b.xt.data(), sizeof(double) * d); }
                else memcpy(X.data() + (size_t)j * d, b.x.data(), sizeof(double) * d);
            }
            if (!any) return PWA_OK;
            pwa_status st = eval();
            if (st != PWA_OK) return st;
#pragma omp parallel for schedule(static) if (Ka >= 4)
            for (int j = 0; j < Ka; ++j) {
                Bfgs &b = fit[act[j]];
                if (b.done) continue;
                memcpy(b.gt.data(), Gr.data() + (size_t)j * d, sizeof(double) * d);
                b.update(F[j], max_iter, gtol);
            }
        }
    };
    // The int8 tensor-core path of the batched call (pwa_batch_path == 2) carries a non-smooth error of ~1e-8 |T| on
    // the gradient and ~1e-9 |L_data| on nll.  Near the minimum the Armijo test then compares noise:
    // the search backtracks ~30 times per iteration and accepts tiny steps by chance.  First stage: on that path three
    // consecutive accepted steps shorter than 2^-10 of the quasi-Newton step end the fit (PWA_FIT_LINE_SEARCH: the
    // resolution of this path is reached).  Second stage: such a fit is continued, from its current point and inverse
    // Hessian, on the FP64 DMMA path ("batch" = 1) until gtol, max_iter or the fp64 resolution; only those fits are
    // evaluated there.
    int32_t path = -1;
    const bool noisy = K > 1 && pwa_batch_path(ctx, &path, nullptr) == PWA_OK && path == 2;
    if (noisy) for (int k = 0; k < K; ++k) fit[k].stall_limit = 3;
    s = lockstep();
    if (s != PWA_OK) return s;
    if (noisy) {
        act.clear();
        for (int k = 0; k < K; ++k) if (fit[k].why == PWA_FIT_LINE_SEARCH && fit[k].iter < max_iter) act.push_back(k);
        int32_t old_opt = 0;
        if (!act.empty() && pwa_get_option(ctx, "batch", &old_opt) == PWA_OK && pwa_set_option(ctx, "batch", 1) == PWA_OK) {
            const int Ka = (int)act.size();
            for (int j = 0; j < Ka; ++j) memcpy(X.data() + (size_t)j * d, fit[act[j]].x.data(), sizeof(double) * d);
            s = eval();
            if (s == PWA_OK) {
                for (int j = 0; j < Ka; ++j) {
                    Bfgs &b = fit[act[j]];
                    b.f = F[j];
                    memcpy(b.g.data(), Gr.data() + (size_t)j * d, sizeof(double) * d);
                    b.done = false; b.why = 0; b.stall_limit = 0; b.small_steps = 0;
                    if (b.gmax() < gtol) { b.done = true; b.why = PWA_FIT_CONVERGED; }
                    else b.direction(false);
                }
                s = lockstep();
            }
            pwa_set_option(ctx, "batch", old_opt);
            if (s != PWA_OK) return s;
        }
    }
    for (int k = 0; k < K; ++k) {
        memcpy(V + (size_t)k * d, fit[k].x.data(), sizeof(double) * d);
        if (nll_out) nll_out[k] = fit[k].f;
        if (n_iter_out) n_iter_out[k] = fit[k].iter;
        if (why_out) why_out[k] = fit[k].why;
    }
    if (n_evals_out) *n_evals_out = evals;
    return worst;
}

pwa_status pwa_minimize_bfgs_floating(pwa_ctx *ctx, double *V, double *mass, double *width, int32_t n_res,
                                      const int32_t *free_res, int32_t n_free, int32_t max_iter, double gtol,
                                      double *nll_out, int32_t *n_iter_out, int32_t *n_evals_out)
{
    return pwa_minimize_bfgs_floating_ex(ctx, V, mass, width, n_res, free_res, n_free, max_iter, gtol, nll_out, n_iter_out,
                                         n_evals_out, nullptr);
}

pwa_status pwa_minimize_bfgs_floating_ex(pwa_ctx *ctx, double *V, double *mass, double *width, int32_t n_res,
                                         const int32_t *free_res, int32_t n_free, int32_t max_iter, double gtol,
                                         double *nll_out, int32_t *n_iter_out, int32_t *n_evals_out, int32_t *why_out)
{
    if (!ctx || !V || !mass || !width || n_res < 1 || n_res > 64 || n_free < 0 || n_free > n_res || (n_free > 0 && !free_res) || max_iter < 0)
        return PWA_ERR_INVALID_ARG;
    for (int i = 0; i < n_free; ++i) {
        if (free_res[i] < 0 || free_res[i] >= n_res) return PWA_ERR_INVALID_ARG;
        for (int j = 0; j < i; ++j) if (free_res[j] == free_res[i]) return PWA_ERR_INVALID_ARG;
    }
    if (n_res != pwa_n_res(ctx)) return PWA_ERR_INVALID_ARG;      // mass / width arrays are sized by the wave map's n_res
    const int n = pwa_n_waves(ctx), d = 2 * n + 2 * n_free;
    // parameter vector: [Re V_0, Im V_0, ..., M_free[0..], G_free[0..]], minimised in SCALED variables u = x / sc:
    // sc = 1 for V, 1 % of the starting mass, 2 % of the starting width (the first step, normalised to |du| = 1,
    // then moves a resonance by at most ~1 %: an unscaled unit step would throw it across its neighbours, and the
    // likelihood has one local minimum per assignment of resonances to peaks)
    std::vector<double> x(d), u(d), sc(d, 1.0), g(d), Mr(mass, mass + n_res), Gr(width, width + n_res), dM(n_res), dG(n_res);
    memcpy(x.data(), V, sizeof(double) * 2 * n);
    int32_t gauge = 0;                               // fixed-phase gauge of V, as in pwa_minimize_bfgs_batch_ex
    if (pwa_get_option(ctx, "fix_phase", &gauge) != PWA_OK) gauge = 0;
    const int ref = gauge - 1;
    if (ref >= 0) pwa_fix_phase_host(n, ref, x.data(), nullptr);
    for (int i = 0; i < n_free; ++i) {
        x[2 * n + i] = mass[free_res[i]]; x[2 * n + n_free + i] = width[free_res[i]];
        sc[2 * n + i] = 0.01 * fabs(mass[free_res[i]]); sc[2 * n + n_free + i] = 0.02 * fabs(width[free_res[i]]);
        if (!(sc[2 * n + i] > 0.0) || !(sc[2 * n + n_free + i] > 0.0)) return PWA_ERR_INVALID_ARG;
    }
    for (int i = 0; i < d; ++i) u[i] = x[i] / sc[i];
    int32_t evals = 0;
    pwa_status worst = PWA_OK;
    bool two_pass = true;
    // f(x), grad f(x); returns +inf for a non-physical trial point (the line search backs off)
    double norm_last = 0.0;                          // Norm of the most recent evaluation
    auto eval = [&](const double *uu, double *f, double *gg) -> pwa_status {
        double parts[2] = {0.0, 0.0};
        std::vector<double> xv(d);
        for (int i = 0; i < d; ++i) xv[i] = uu[i] * sc[i];
        const double *xx = xv.data();
        for (int i = 0; i < n_free; ++i) {
            Mr[free_res[i]] = xx[2 * n + i]; Gr[free_res[i]] = xx[2 * n + n_free + i];
            if (!(Mr[free_res[i]] > 0.0) || !(Gr[free_res[i]] > 0.0)) { *f = INFINITY; return PWA_OK; }
        }
        pwa_status s = PWA_OK;
        if (two_pass) {                                   // one evaluation = two streaming passes (pwa.h)
            s = pwa_nll_grad_floating(ctx, xx, Mr.data(), Gr.data(), f, gg, dM.data(), dG.data(), parts);
            if (s == PWA_ERR_UNSUPPORTED) two_pass = false;
            else {
                evals += 1;
                norm_last = parts[1];
                if (s == PWA_WARN_NONFINITE) { worst = s; s = PWA_OK; }
                if (s != PWA_OK) return s;
                for (int i = 0; i < n_free; ++i) { gg[2 * n + i] = dM[free_res[i]]; gg[2 * n + n_free + i] = dG[free_res[i]]; }
                for (int i = 0; i < d; ++i) gg[i] *= sc[i];
                if (ref >= 0) gg[2 * ref + 1] = 0.0;
                return PWA_OK;
            }
        }
        s = pwa_set_resonances(ctx, Mr.data(), Gr.data());
        if (s != PWA_OK) return s;
        s = pwa_build_norm(ctx, nullptr);
        if (s != PWA_OK) return s;
        s = pwa_nll_grad(ctx, xx, f, gg, parts);
        evals += 1;
        norm_last = parts[1];
        if (s == PWA_WARN_NONFINITE) { worst = s; s = PWA_OK; }
        if (s != PWA_OK) return s;
        if (n_free > 0) {
            s = pwa_res_grad(ctx, xx, dM.data(), dG.data());
            if (s != PWA_OK) return s;
            for (int i = 0; i < n_free; ++i) { gg[2 * n + i] = dM[free_res[i]]; gg[2 * n + n_free + i] = dG[free_res[i]]; }
        }
        for (int i = 0; i < d; ++i) gg[i] *= sc[i];       // d f / d u
        if (ref >= 0) gg[2 * ref + 1] = 0.0;
        return PWA_OK;
    };
    Bfgs fit;
    double f0 = 0.0;
    pwa_status s = eval(u.data(), &f0, g.data());
    if (s != PWA_OK) return s;
    if (!isfinite(f0)) return PWA_ERR_INVALID_ARG;      // the starting point itself must be physical
    {   // Euler prescale of V (see pwa_minimize_bfgs_batch_ex): s^2 = N_data / Norm at the starting resonance parameters
        int32_t lik = 0;
        const double n_data = (double)pwa_n_events(ctx, PWA_DATA);
        if (pwa_get_option(ctx, "likelihood", &lik) == PWA_OK && lik == 0 && n_data > 0.0 && norm_last > 0.0 && isfinite(norm_last) && max_iter > 0) {
            const double scv = sqrt(n_data / norm_last);
            for (int i = 0; i < 2 * n; ++i) u[i] *= scv;           // sc = 1 for the V components
            s = eval(u.data(), &f0, g.data());
            if (s != PWA_OK) return s;
            if (!isfinite(f0)) return PWA_ERR_INVALID_ARG;
        }
    }
    fit.init(d, u.data());
    // the likelihood has one local minimum per assignment of resonances to peaks: an iteration may move a mass by at most
    // 3 % and a width by at most 6 % of its starting value (3 scaled units), so that the fit stays in the basin it started in
    fit.cap.assign(d, 0.0);
    for (int i = 2 * n; i < d; ++i) fit.cap[i] = 3.0;
    fit.f = f0; fit.g = g;
    if (fit.gmax() < gtol) { fit.done = true; fit.why = PWA_FIT_CONVERGED; }
    else if (max_iter == 0) { fit.done = true; fit.why = PWA_FIT_MAX_ITER; }
    else fit.direction(true);
    while (!fit.done) {
        fit.trial();
        double ft = 0.0;
        s = eval(fit.xt.data(), &ft, fit.gt.data());
        if (s != PWA_OK) return s;
        fit.update(ft, max_iter, gtol);
    }
    for (int i = 0; i < d; ++i) x[i] = fit.x[i] * sc[i];
    memcpy(V, x.data(), sizeof(double) * 2 * n);
    for (int i = 0; i < n_free; ++i) { mass[free_res[i]] = x[2 * n + i]; width[free_res[i]] = x[2 * n + n_free + i]; }
    // leave the context at the fitted point (M valid for it)
    for (int i = 0; i < n_free; ++i) { Mr[free_res[i]] = mass[free_res[i]]; Gr[free_res[i]] = width[free_res[i]]; }
    s = pwa_set_resonances(ctx, Mr.data(), Gr.data());
    if (s != PWA_OK) return s;
    s = pwa_build_norm(ctx, nullptr);
    if (s != PWA_OK) return s;
    if (nll_out) *nll_out = fit.f;
    if (n_iter_out) *n_iter_out = fit.iter;
    if (n_evals_out) *n_evals_out = evals;
    if (why_out) *why_out = fit.why;
    return worst;
}

}  // extern "C"
