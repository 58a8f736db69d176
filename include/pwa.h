/*
 * pwa.h — C ABI of libpwa.so: the per-iteration extended log-likelihood and gradient of an
 * unbinned partial-wave-analysis fit (arXiv 1108.5882, N. Berger, "Partial Wave Analysis
 * using Graphics Cards"), computed on one NVIDIA B200 (sm_100a).
 *
 * Citations: "P:n" = line n of the paper text; "C<k>" = reading k in DESIGN.md
 * section 3 (where the paper is silent).  Notation:
 *   n waves (index a), N data events (i), N_acc accepted MC events (j), N_gen generated MC;
 *   A[i][a] = A_a(Omega_i), B[j][a] = A_a(Omega_j);  V_a = x_a + i y_a;
 *   S_i = sum_a V_a A_ia,  I_i = |S_i|^2                                  (eq. 1)
 *   L_data = sum_i ln I_i                                                  (eq. 3 first term)
 *   Norm   = (1/N_gen) sum_j |sum_a V_a B_ja|^2 = V^H M V,  M = B^H B / N_gen   (eq. 3 second term; C1)
 *   nll    = -(L_data - Norm)                                              (P:55 fn. 3)
 *   T_a    = sum_i A_ia / S_i;   grad_a = d nll/d x_a + i d nll/d y_a = -2 conj(T_a) + 2 (M V)_a   (C6)
 *
 * General rules.  All symbols are extern "C"; no exception, abort() or stdout output
 * crosses the ABI.  Every call returns a pwa_status; on PWA_ERR_* the outputs are
 * untouched and pwa_last_error() describes the failure.  The library never frees or keeps
 * caller memory except as stated for PWA_BORROW.  One context = one CUDA stream = one host
 * thread at a time.  All scratch is owned by the context.  Everything pwa_nll_grad and pwa_data_term_enqueue need
 * (per-block partial slots, result records, V staging) is allocated in pwa_create; the work space of pwa_build_norm,
 * pwa_nll_grad_batch and pwa_fumili_hessian is allocated by the first call of that kind (it grows only when a later
 * call needs more: a larger K), so the steady-state calls of a fit never allocate.  There is no CPU fallback: without a CUDA device
 * pwa_create fails with PWA_ERR_CUDA.
 *
 * Pointer kinds are stated per argument: HOST = ordinary host memory, DEVICE = CUDA device
 * memory of the context's device, ANY = either (detected with cudaPointerGetAttributes).
 * Complex numbers are interleaved (re, im).  Matrices are row-major.
 */
#ifndef PWA_H_
#define PWA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pwa_ctx pwa_ctx; /* opaque, library-owned */

typedef enum {
    PWA_OK = 0,
    PWA_ERR_INVALID_ARG = 1,
    PWA_ERR_STATE = 2,        /* call order wrong: data not uploaded, M missing or stale, ... */
    PWA_ERR_OOM = 3,
    PWA_ERR_CUDA = 4,
    PWA_ERR_UNSUPPORTED = 5,
    PWA_WARN_NONFINITE = 6    /* results written, but some I_i was 0 or non-finite (C14) */
} pwa_status;

typedef enum { PWA_F64 = 0, PWA_F32 = 1 } pwa_dtype;   /* amplitude STORAGE type (C16) */
typedef enum { PWA_DATA = 0, PWA_MC = 1 } pwa_sample;

#define PWA_COPY   0u   /* library copies the events into its own device buffer (default) */
#define PWA_BORROW 1u   /* DEVICE pointer in native layout is used in place; caller keeps it
                           alive and unchanged until the next upload of that sample or destroy */

/* ---- life cycle ----------------------------------------------------------------------- */

/* n_waves >= 1.  storage: element type of every amplitude array given to this context
 * (arithmetic and accumulation are always fp64).  device: CUDA ordinal.
 * cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL for
 * the legacy default stream.  All work of the context is enqueued on that stream.       */
pwa_status pwa_create(pwa_ctx **out, int32_t n_waves, pwa_dtype storage, int32_t device,
                      void *cuda_stream);
void pwa_destroy(pwa_ctx *ctx);                       /* NULL-safe; frees library memory only */
const char *pwa_last_error(const pwa_ctx *ctx);       /* ctx-owned string, valid until next call */
const char *pwa_status_string(pwa_status s);          /* static string */

/* ---- event upload --------------------------------------------------------------------- */

/* Constant-resonance mode (amplitudes pre-calculated once per fit).
 * amps: ANY pointer, row-major [n_events][n_waves] complex, element type = ctx storage.
 * n_generated: N_gen of eq. 3, used for which == PWA_MC only and must then be
 * >= n_events (C9); ignored for PWA_DATA.  n_events may be 0.
 * flags: PWA_COPY or PWA_BORROW (BORROW requires a DEVICE pointer, 16-byte aligned).
 * Uploading PWA_MC marks M stale.                                                        */
pwa_status pwa_upload_events(pwa_ctx *ctx, pwa_sample which, const void *amps,
                             int64_t n_events, int64_t n_generated, uint32_t flags);

/* Floating-resonance mode (when masses/widths float nothing can be pre-calculated):
 *   A_ia = BW(mass_i; M_r(a), G_r(a)) * ang[i][s(a)],  BW(m; M, G) = 1/(M^2 - m^2 - i M G)  (C3)
 * and the Breit-Wigner factors are recomputed inside every kernel that reads the sample.
 * mass: ANY, [n_events] doubles (always fp64).  ang: ANY, [n_events][n_ang] complex of the
 * ctx storage type.  1 <= n_ang <= 4.  Needs pwa_set_wave_map + pwa_set_resonances before
 * any evaluation.                                                                        */
pwa_status pwa_upload_events_factored(pwa_ctx *ctx, pwa_sample which, const double *mass,
                                      const void *ang, int32_t n_ang, int64_t n_events,
                                      int64_t n_generated, uint32_t flags);

/* Optional per-event weights.  MC: a sample that was not
 * generated evenly in phase space is re-weighted (P:37 fn. 2): M_ab = (1/N_gen) sum_j w_j conj(B_ja) B_jb.
 * DATA (reading: weighted unbinned likelihood, e.g. side-band subtraction with negative weights):
 * L_data = sum_i w_i ln I_i, T_a = sum_i w_i A_ia / S_i.  w: ANY, [n_events] doubles of the sample
 * uploaded LAST for `which` (a new upload drops the weights); NULL removes them.  flags as for uploads.
 * Setting MC weights marks M stale.  Weighted samples use the FP64 paths (per-lane streaming kernel,
 * DMMA Gram kernel); weights are not supported with factored uploads or n > 64 (PWA_ERR_UNSUPPORTED
 * at evaluation).                                                                                  */
pwa_status pwa_set_weights(pwa_ctx *ctx, pwa_sample which, const double *w, uint32_t flags);

/* res_of_wave[a] in [0, n_res), ang_of_wave[a] in [0, n_ang): HOST int32 [n_waves].
 * 1 <= n_res <= 64.  Each (resonance, angular structure) pair may belong to at most one
 * wave.                                                                                   */
pwa_status pwa_set_wave_map(pwa_ctx *ctx, int32_t n_res, const int32_t *res_of_wave,
                            const int32_t *ang_of_wave);

/* mass0, width0: HOST [n_res] doubles (GeV).  Marks M stale (it must be rebuilt).  */
pwa_status pwa_set_resonances(pwa_ctx *ctx, const double *mass0, const double *width0);

/* ---- normalisation matrix (P:41 inner bracket) ----------------------------------- */

/* Builds M = B^H B / N_gen over the uploaded MC sample (Breit-Wigner fused in factored
 * mode) and keeps it on the device for the evaluation calls.  M_out: optional HOST buffer
 * [n][n][2] doubles, M_out[a][b] = M_ab = (1/N_gen) sum_j conj(B_ja) B_jb (C1); may be NULL.
 * Synchronous when M_out != NULL.  PWA_ERR_STATE if no MC sample was uploaded.           */
pwa_status pwa_build_norm(pwa_ctx *ctx, double *M_out);

/* A-priori bound on max_ab |M_ab(library) - M_ab(exact fp64 sum over the stored amplitudes)| of the
 * most recent pwa_build_norm.  The FP64 paths only carry summation rounding (reported as 0); the
 * int8 tensor-core path for fp32-stored samples (fixed-point digit planes, exact integer
 * accumulation, low orders truncated: DESIGN.md section 6.6) reports its quantisation + truncation
 * bound in the units of M.  *which_path (may be NULL): 0 = FP64 path, 1 = int8 tcgen05 path, 3 = its three-plane
 * variant ("norm" = 3).                                                                                 */
pwa_status pwa_norm_error_bound(pwa_ctx *ctx, double *bound, int32_t *which_path);

/* Installs an externally computed M (HOST [n][n][2]), e.g. the sum over ranks of per-shard
 * matrices in an event-sharded multi-GPU run.                                      */
pwa_status pwa_set_norm(pwa_ctx *ctx, const double *M);

/* ---- evaluation: the per-iteration hot path -------------------------------------------- */

/* V: HOST [n][2] doubles.  Outputs (HOST): *nll = -(L_data - V^H M V);
 * grad[n][2] = (d nll / d Re V_a, d nll / d Im V_a);  parts (may be NULL): [0] = L_data,
 * [1] = Norm.  One pass over the data amplitudes in HBM; synchronous (returns after the
 * results are in host memory: the kernel's finishing block writes them into pinned host memory and
 * raises a flag the call polls, so no device-to-host copy is enqueued).  PWA_ERR_STATE if DATA is missing or M is missing / stale.
 * PWA_WARN_NONFINITE if some I_i was 0 or not finite (IEEE values are still written).     */
pwa_status pwa_nll_grad(pwa_ctx *ctx, const double *V, double *nll, double *grad,
                        double *parts);

/* K starting points in one pass over the data.  V: HOST [K][n][2];
 * nll: [K]; grad: [K][n][2]; parts: [K][2] or NULL.  Column k equals pwa_nll_grad(V_k)
 * to floating-point tolerance (not necessarily bitwise).  1 <= K <= 1024.                */
pwa_status pwa_nll_grad_batch(pwa_ctx *ctx, int32_t K, const double *V, double *nll,
                              double *grad, double *parts);

/* Which kernel family served the most recent pwa_nll_grad_batch / _batch_enqueue:
 * 0 = K passes of the streaming data-term kernel, 1 = chained FP64 DMMA GEMMs (batch_dmma.cu),
 * 2 = chained int8 tcgen05 GEMMs with exact int32 accumulation (batch_i8.cu, DESIGN.md section 6.7:
 * fp32-stored constant-resonance data sample, n = 64, no event weights; default for K >= 8 and
 * >= 32768 events).  *err_rel (may be NULL): for path 2 the a-priori estimate of the relative error
 * of each term A_ia / S_ik entering the gradient sums (independent over events: the norm-wise error of
 * the summed gradient is smaller by about 1 / sqrt(N_data)), else 0.  PWA_ERR_STATE before the first
 * batched call.                                                                                  */
pwa_status pwa_batch_path(pwa_ctx *ctx, int32_t *which_path, double *err_rel);

/* Asynchronous pair: enqueue one evaluation (V is copied before return) / wait and fetch
 * the results of the most recent enqueue.  Used for device-side timing.                  */
pwa_status pwa_nll_grad_enqueue(pwa_ctx *ctx, const double *V);
pwa_status pwa_nll_grad_batch_enqueue(pwa_ctx *ctx, int32_t K, const double *V);
pwa_status pwa_fetch(pwa_ctx *ctx, int32_t K, double *nll, double *grad, double *parts);

/* Data term only, for event-sharded multi-GPU runs ("treat different subsets of
 * events on different ... machines ... then ... perform a synthesis"): enqueues one pass
 * and writes out_dev (DEVICE, [2 + 2n] doubles) = { L_data, n_nonfinite, Re T_0, Im T_0,
 * ... } of THIS context's events.  The caller sums out_dev over ranks and finishes with
 * pwa_assemble_host.  Asynchronous.                                                      */
pwa_status pwa_data_term_enqueue(pwa_ctx *ctx, const double *V, double *out_dev);

/* The same record WITHOUT any allocation and without a context, for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it): steps A2 - A5 (eq. 1; eq. 3 first term, P:41;
 * fp64 reduction) over amps_dev (DEVICE, row-major [n_events][n_waves] complex interleaved, element type
 * `storage`, caller-owned, not kept) at V (HOST [n_waves][2], passed to the kernel by value) -> out_dev (DEVICE,
 * [2 + 2 n_waves] doubles = { L_data, n_nonfinite, Re T_0, Im T_0, ... }).  Asynchronous on cuda_stream (cudaStream_t,
 * may be 0) of `device`.  The per-block partial sums of the fixed-order reduction live in ONE static device array of
 * 1 065 216 bytes that every GPU holds from the moment it loads the library until the process exits; it limits the
 * call to n_waves <= PWA_STATIC_MAX_WAVES (PWA_ERR_UNSUPPORTED beyond, with the reason in errbuf; any n_events >= 0 is
 * served, the grid is capped at 1024 blocks).  The call issues one 256-byte cudaMemsetAsync and one kernel launch and
 * calls no cudaMalloc / cudaFree / allocating library routine; its first call on a device looks up the array's address
 * (do that once before a capture).  Every call shares the array: calls that OVERLAP on the GPU (different streams, or
 * several host threads) race and return wrong sums; calls on one stream are ordered and safe.  A plain lane-group
 * streaming kernel (no TMA, no event weights, constant resonances only; amps_dev 16-byte aligned): ~1.3 TB/s at
 * 5e6 events x 64 waves fp32, about a fifth of the context path's rate; bitwise reproducible for a fixed shape.  errbuf (HOST, errbuf_len bytes, may be NULL) receives the error text.              */
#define PWA_STATIC_MAX_WAVES 64
pwa_status pwa_data_term_static(int32_t device, void *cuda_stream, pwa_dtype storage, int32_t n_waves,
                                const void *amps_dev, int64_t n_events, const double *V, double *out_dev,
                                char *errbuf, int32_t errbuf_len);

/* Host-only step A7: Norm = V^H M V, nll = -(L_data - Norm), grad = -2 conj(T) + 2 M V.
 * All pointers HOST; T [n][2], M [n][n][2], V [n][2]; parts [2] or NULL.  No GPU needed. */
pwa_status pwa_assemble_host(int32_t n_waves, double L_data, const double *T, const double *M,
                             const double *V, double *nll, double *grad, double *parts);

/* Event-sharded runs, one context per shard (rank).  All three are host-side synthesis steps with the
 * shards added in index order r = 0 .. R-1, so every rank that is given the same gathered arrays obtains the
 * same bits (a tree all-reduce would not fix the order).
 * pwa_norm_sums: G = B^H B over THIS context's MC events without the 1/N_gen (N_gen times the M of the most
 *   recent pwa_build_norm), HOST [n][n][2], and this shard's N_gen.  PWA_ERR_STATE without a valid M.
 * pwa_combine_norm_host: M_out = (sum_r G_r) / (sum_r N_gen,r)  (eq. 3 second term, over all shards);
 *   G HOST [R][n][n][2], n_gen HOST [R], M_out HOST [n][n][2] (for pwa_set_norm), *n_gen_total (may be NULL) the
 *   summed N_gen.  No GPU needed.
 * pwa_assemble_host_shards: terms HOST [R][2 + 2n], the records pwa_data_term_enqueue wrote on the R shards;
 *   adds them and performs step A7 as pwa_assemble_host (likelihood = 0) or pwa_assemble_host_eq2 (likelihood = 1,
 *   n_data = N_data of ALL shards).  PWA_WARN_NONFINITE if any shard counted a non-finite event.  No GPU needed. */
pwa_status pwa_norm_sums(pwa_ctx *ctx, double *G_out, int64_t *n_gen_out);
pwa_status pwa_combine_norm_host(int32_t n_waves, int32_t R, const double *G, const int64_t *n_gen, double *M_out,
                                 int64_t *n_gen_total);
pwa_status pwa_assemble_host_shards(int32_t n_waves, int32_t R, const double *terms, const double *M, const double *V,
                                    int32_t likelihood, double n_data, double *nll, double *grad, double *parts);

/* Fumili-style approximate Hessian of nll at V (Minuit / Fumili; "most of the computing time
 * is spent on ... error calculations"), DESIGN.md section 13:
 *   H = sum_i u_i u_i^T  (+ Hess(Norm) if with_norm != 0),   u_i = d ln I_i / d(x_0, y_0, x_1, ...)
 *     = (2 Re t_i0, -2 Im t_i0, ...),  t_ia = A_ia / S_i;  Hess(Norm) = 2 [[Re M, -Im M], [Im M, Re M]].
 * One extra pass over the DATA sample: a second dense contraction (the Gram matrix of the rows
 * A_i / S_i) on the FP64 tensor cores.  V: HOST [n][2].  H: HOST [2n][2n] doubles, row-major,
 * parameter order as in grad; exactly symmetric, positive semi-definite without the norm part.
 * n <= 64.  PWA_ERR_STATE if DATA (or, with_norm, M) is missing.  Synchronous.                  */
pwa_status pwa_fumili_hessian(pwa_ctx *ctx, const double *V, double *H, int32_t with_norm);

/* eq. 2 form of step A7: the likelihood normalised by the MC integral instead of the
 * extended form of eq. 3 (reading C2):  nll2 = -L_data + N_data ln Norm,
 * grad2 = -2 conj(T) + (2 N_data / Norm) M V.  Invariant under V -> s V.  Host only; same
 * argument meaning as pwa_assemble_host, n_data = N_data > 0.  On the device the same form is
 * selected for pwa_nll_grad / pwa_nll_grad_batch with pwa_set_option(ctx, "likelihood", 1); N_data is then the
 * number of data events, or the sum of their weights when pwa_set_weights attached some (the weighted
 * normalised likelihood -sum_i w_i ln I_i + (sum_i w_i) ln Norm, which keeps the invariance under V -> s V). */
pwa_status pwa_assemble_host_eq2(int32_t n_waves, double n_data, double L_data, const double *T,
                                 const double *M, const double *V, double *nll, double *grad,
                                 double *parts);

/* Polar parametrisation V_a = r_a exp(i phi_a), host only.  pwa_grad_to_polar: chain
 * rule on a Cartesian gradient grad[n][2] at V[n][2] -> grad_polar[n][2] = (d/dr_a, d/dphi_a)
 * (at r_a = 0 the radial direction is taken along the real axis).  pwa_polar_to_cartesian:
 * r_phi[n][2] = (r_a, phi_a) -> V[n][2].                                                        */
pwa_status pwa_grad_to_polar(int32_t n_waves, const double *V, const double *grad, double *grad_polar);
pwa_status pwa_polar_to_cartesian(int32_t n_waves, const double *r_phi, double *V);

/* Fixed-phase gauge, host only.  nll (eq. 3 and eq. 2) depends on V only up to a common phase:
 * |S_i| and V^dagger M V do not change under V -> exp(i a) V, which leaves every fit one flat direction.  The gauge
 * "wave ref_wave is real and non-negative" removes it.  pwa_fix_phase_host turns V[n][2] IN PLACE by
 * exp(-i arg V_ref) (exact complex multiplication by conj(V_ref) / |V_ref|; Im V_ref is set to exactly 0); when grad
 * is not NULL the Cartesian gradient grad[n][2], read as g_a = d/dRe V_a + i d/dIm V_a, is turned by the same factor
 * (it is then the gradient at the turned V) and its component d/dIm V_ref, the parameter the gauge fixes, is set to 0.
 * V_ref = 0 leaves V and grad unturned (only the component is zeroed).  PWA_ERR_INVALID_ARG for ref_wave outside
 * [0, n_waves).  The minimisers apply the gauge themselves with pwa_set_option(ctx, "fix_phase", ref_wave + 1).     */
pwa_status pwa_fix_phase_host(int32_t n_waves, int32_t ref_wave, double *V, double *grad);

/* Floating mode: gradient of nll w.r.t. the resonance parameters at the current
 * (mass0, width0) and the given V (reading A9):  d nll / d M_r and d nll / d G_r, HOST
 * [n_res] each (n_res of pwa_set_wave_map: see pwa_n_res).  Needs factored DATA and MC uploads.  One extra pass
 * over data and MC.  With "likelihood" = 1 the eq. 2 form is differentiated:
 * -d L_data / d theta + (N_data / Norm) d Norm / d theta, Norm evaluated by the same MC pass.                  */
pwa_status pwa_res_grad(pwa_ctx *ctx, const double *V, double *dnll_dmass, double *dnll_dwidth);

/* One evaluation of a floating-resonance fit in TWO streaming passes (with floating masses and widths every
 * evaluation has its own Breit-Wigner factors, so a matrix M built for it would be used exactly once; Norm, its
 * gradient and all resonance derivatives are then cheaper as the explicit MC sum of eq. 3, O(N_acc n) instead
 * of O(N_acc n^2)):
 *   MC pass:   Norm = (1/N_gen) sum_j |S_j|^2,  2 (M V)_a = (2/N_gen) sum_j conj(B_ja) S_j,  d Norm / d(M_r, G_r)
 *   data pass: L_data, T_a, d L_data / d(M_r, G_r)
 * both with the Breit-Wigner factors recomputed in registers from (mass, ang).  Sets the resonance parameters to
 * (mass0, width0) (HOST [n_res], as pwa_set_resonances: a previously built M becomes stale) and returns
 * nll, grad[n][2], d nll / d M_r, d nll / d G_r (HOST [n_res] each), parts = {L_data, Norm} (may be NULL); the same
 * numbers as pwa_build_norm + pwa_nll_grad + pwa_res_grad to rounding.  Honours "likelihood".  Needs factored DATA and
 * MC uploads with the same n_ang, a wave map, and n + n_res * n_ang <= 64 (PWA_ERR_UNSUPPORTED otherwise: use the three
 * calls).  Synchronous.                                                                                          */
pwa_status pwa_nll_grad_floating(pwa_ctx *ctx, const double *V, const double *mass0, const double *width0,
                                 double *nll, double *grad, double *dnll_dmass, double *dnll_dwidth, double *parts);

/* ---- host minimiser (a quasi-Newton in real parameters stays on the host) --- */

/* All three minimisers first rescale the starting V by s = sqrt(N_data / Norm(V)) in the eq. 3 form: along V -> s V the
 * extended likelihood is L_data + N ln s^2 - s^2 Norm, so the optimal scale is known in closed form.
 * Plain BFGS with backtracking line search on the 2n reals of V (constant-resonance mode).
 * V_inout: HOST [n][2], start in / result out.  Stops after max_iter iterations, when
 * max|grad| < gtol, or when the line search is exhausted.  nll_out, n_iter_out, n_evals_out may be NULL. */
pwa_status pwa_minimize_bfgs(pwa_ctx *ctx, double *V_inout, int32_t max_iter, double gtol,
                             double *nll_out, int32_t *n_iter_out, int32_t *n_evals_out);

/* K independent BFGS fits run in lock-step on pwa_nll_grad_batch.  V_inout [K][n][2].
 * The evaluations take the batched call's DEFAULT path (pwa_batch_path): for fp32-stored samples with n = 64,
 * K >= 8 and >= 32768 events that is the int8 tcgen05 path, whose gradient carries a non-smooth error floor of
 * about 1e-8 |T| (norm-wise): a gtol below that floor cannot be reached and such a fit ends
 * with PWA_FIT_LINE_SEARCH or PWA_FIT_MAX_ITER; pwa_set_option(ctx, "batch", 1) (FP64 DMMA) gives the last
 * digits; pwa_minimize_bfgs_batch does so itself: fits whose line search ran out of resolution on the int8 path are
 * continued (same point, same inverse Hessian) on the FP64 DMMA path, and only those fits are evaluated there.
 * The _ex form also reports, per fit, the iterations done and why it stopped (either may be NULL). */
#define PWA_FIT_CONVERGED   0   /* max|grad| < gtol */
#define PWA_FIT_MAX_ITER    1   /* max_iter iterations done */
#define PWA_FIT_LINE_SEARCH 2   /* backtracking exhausted (step < 1e-20): the resolution of nll / its gradient is reached */
pwa_status pwa_minimize_bfgs_batch(pwa_ctx *ctx, int32_t K, double *V_inout, int32_t max_iter,
                                   double gtol, double *nll_out /* [K] */,
                                   int32_t *n_evals_out);
pwa_status pwa_minimize_bfgs_batch_ex(pwa_ctx *ctx, int32_t K, double *V_inout, int32_t max_iter, double gtol,
                                      double *nll_out /* [K] */, int32_t *n_iter_out /* [K] */,
                                      int32_t *why_out /* [K]: PWA_FIT_* */, int32_t *n_evals_out);

/* Floating-resonance fit (configs[3]; with floating masses and widths nothing can be pre-calculated, so
 * EVERY evaluation re-evaluates the Breit-Wigner factors and rebuilds M): BFGS over the 2 n_waves Cartesian reals
 * of V and the masses and widths of the n_free resonances listed in free_res (HOST int32 [n_free], distinct
 * indices in [0, n_res)).  One evaluation = pwa_nll_grad_floating (two passes), or, where that is not supported,
 * pwa_set_resonances + pwa_build_norm + pwa_nll_grad + pwa_res_grad (four passes).  V_inout: HOST [n][2]; mass_inout,
 * width_inout: HOST [n_res], all resonances (the fixed ones are read, the free ones updated).  A trial point with a
 * non-positive mass or width is rejected by the line search.  Needs factored DATA and MC uploads and a wave map.
 * n_res must equal pwa_n_res(ctx) (PWA_ERR_INVALID_ARG otherwise).  nll_out, n_iter_out, n_evals_out, why_out
 * (PWA_FIT_*) may be NULL.  Honours "likelihood" (eq. 2 / eq. 3) in the objective AND in all gradient components. */
pwa_status pwa_minimize_bfgs_floating(pwa_ctx *ctx, double *V_inout, double *mass_inout, double *width_inout,
                                      int32_t n_res, const int32_t *free_res, int32_t n_free, int32_t max_iter,
                                      double gtol, double *nll_out, int32_t *n_iter_out, int32_t *n_evals_out);
pwa_status pwa_minimize_bfgs_floating_ex(pwa_ctx *ctx, double *V_inout, double *mass_inout, double *width_inout,
                                         int32_t n_res, const int32_t *free_res, int32_t n_free, int32_t max_iter,
                                         double gtol, double *nll_out, int32_t *n_iter_out, int32_t *n_evals_out,
                                         int32_t *why_out);

/* ---- introspection / measurement ------------------------------------------------------- */

/* n_waves / storage type the context was created with; n_res of the wave map (0 before pwa_set_wave_map);
 * number of events of the sample uploaded last (-1: none).  The binding validates array shapes against these. */
int32_t pwa_n_waves(const pwa_ctx *ctx);
int32_t pwa_n_res(const pwa_ctx *ctx);
pwa_dtype pwa_storage(const pwa_ctx *ctx);
int64_t pwa_n_events(const pwa_ctx *ctx, pwa_sample which);

/* Number of CUDA kernels this context has launched since creation.                        */
uint64_t pwa_launch_count(const pwa_ctx *ctx);

/* Waits for all enqueued work of the context.                                             */
pwa_status pwa_sync(pwa_ctx *ctx);

/* Selects a kernel family (0 = default).  Returns PWA_ERR_INVALID_ARG for unknown keys.
 * Keys: "data_term", "norm", "batch", "l2_resident_mb", "likelihood", "resident", "fix_phase".
 * "data_term": 0 = default (TMA-tiled streaming kernel where the row is 128 .. 1024 bytes and the sample carries no
 * event weights, else the per-lane streaming kernel), 20 = per-lane kernel, 98 = default without programmatic
 * dependent launch, 99 = generic kernel (any n).
 * "norm": 0 = default (int8 tcgen05 path for fp32-stored constant-resonance samples of >= 65536 events, else
 * FP64 DMMA), 1 = FP64 DMMA, 2 = int8 tcgen05 path whenever the shape allows, 3 = the same with THREE digit planes
 * (24 instead of 32 bits below each column's maximum, 4 instead of 7 digit-pair products per step: faster, and
 * pwa_norm_error_bound then reports a bound ~2^9 times larger, typically above the 1e-6 bar of fp32 storage although
 * the measured error stays ~1e-9 of max|M|; opt-in, never the default), 99 = generic CUDA-core kernel.
 * "batch": 0 = default (see pwa_batch_path), 1 = FP64 DMMA GEMMs for any K, 2 = int8 tcgen05 GEMMs
 * whenever the shape allows, 99 = K passes of the streaming kernel.
 * "l2_resident_mb": MB of the head of the DATA sample that the streaming data term loads with the L2 evict_last
 * policy (the rest: evict_first), so that it stays in L2 from one evaluation to the next; -1 = automatic (48 MB for
 * samples between 64 MB and 1 GiB, else plain loads), 0 = plain loads, up to 120.
 * "likelihood": 0 = eq. 3 extended form (default), 1 = eq. 2 normalised form (see
 * pwa_assemble_host_eq2); applies to pwa_nll_grad, pwa_nll_grad_batch, pwa_res_grad and the minimisers.
 * "fix_phase": 0 = the minimisers leave all 2n real parameters free (default); k in 1 .. n = pwa_minimize_bfgs,
 * pwa_minimize_bfgs_batch(_ex) and pwa_minimize_bfgs_floating(_ex) fit in the gauge Im V_(k-1) = 0, Re V_(k-1) >= 0 at
 * the start (pwa_fix_phase_host on every starting point, the gauge component of every gradient set to 0: 2n - 1 free
 * real parameters per fit, the returned V has Im V_(k-1) = 0 exactly).  Evaluation calls are not affected.
 * "resident": 0 = every evaluation is a kernel launch (default); 1 = pwa_nll_grad evaluates through a RESIDENT grid
 * (below ~1e5 events an iteration costs latency, not bandwidth): the default data-term kernel is
 * launched once, stays on the GPU and takes V / returns the record through tagged 8-byte words in pinned host memory,
 * so that an evaluation costs two PCIe round trips and no launch.  Results are bitwise those of the launched
 * evaluation (same grid, same tiles per block, same reduction order).  Served: n in {4, 8, 16, 32, 64},
 * unweighted, constant resonances, "data_term" 0; anything else evaluates by launches under the option.  While
 * the grid is resident it occupies every SM of the device (other streams of the process wait behind it) and the
 * calling thread spins in pwa_nll_grad; every other entry point of the context that enqueues work or changes what
 * the grid reads (uploads, weights, norm, options, batch / enqueue / minimiser calls, pwa_sync, pwa_destroy) ends
 * the grid first, and the next pwa_nll_grad starts it again (one launch).  A grid that sees no command for ~2 s
 * ends by itself.  Meant for a fit loop of single evaluations on a small sample; leave it off otherwise.  Under a
 * tool that makes kernel launches synchronous (ncu) the launch cannot return while the grid waits for its first
 * command: pwa_nll_grad then fails with PWA_ERR_CUDA after a few restarts (~10 s) instead of hanging.               */
pwa_status pwa_set_option(pwa_ctx *ctx, const char *key, int32_t value);
pwa_status pwa_get_option(pwa_ctx *ctx, const char *key, int32_t *value);   /* current value of a pwa_set_option key */

/* Register-resident peak probes used as roofline denominators:
 * which = 0: fp64 FMA (result TFLOP/s), 1: fp64 mma.sync m8n8k4 (TFLOP/s),
 * 2: HBM read-only stream over `bytes` of scratch (GB/s), 3 .. 6: tcgen05.mma.kind::i8 with M = 128, K = 32 and
 * N = 256 / 128 / 64 / 32, operands in shared memory (int8 Top/s, all SMs), 7: TMEM reads (tcgen05.ld 32x32b.x16 by
 * 16 warps per SM, GB/s), 8: overlap probe: one warp issues a stream of tcgen05.mma.kind::i8 (M = N = 128) while 16 (or,
 * with bit 6 of `bytes`, the 12 that do not share the issuer's scheduler) other warps run one kind of epilogue work;
 * `bytes` = mode + 16 (MMAs on) + 32 (epilogue work on) + 64 (keep the issuer's scheduler free), mode 0 = fp64 FMA,
 * 1 = tcgen05.ld, 2 = st.shared.v4, 3 = integer multiply-add, 4 = ld.shared.v4, 5 = fp32 FMA, 6 = 2 fp64 FMA among 6
 * integer chains, 7 = a stream of 16-byte global loads (3.6 GB of scratch), 8 = WINDOWS: the warps alternate, together,
 * between a window of fp64 FMA chains and one of integer chains (window length in fp64 iterations in bits 8 .. 23 of
 * `bytes`, default 64; bit 7: the integer window comes first); result = milliseconds (compare MMAs alone, the work alone and both: DESIGN.md section 6.7 has the
 * outcome: fp64 arithmetic does not overlap with the int8 MMAs at all).  Synchronous; result HOST.                  */
pwa_status pwa_microbench(pwa_ctx *ctx, int32_t which, int64_t bytes, double *result);

#ifdef __cplusplus
}
#endif
#endif /* PWA_H_ */
