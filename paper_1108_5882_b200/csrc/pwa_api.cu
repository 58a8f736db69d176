// pwa_api.cu — the C ABI of include/pwa.h: context, uploads, call-order checks and the
// host side of each evaluation (argument marshalling and one launch; the finishing block of the
// kernel writes the result record into device-mapped pinned host memory, so no D2H copy is enqueued).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "pwa_internal.h"

namespace pwa {

pwa_status fail(pwa_ctx *ctx, pwa_status s, const std::string &msg)
{
    if (ctx) ctx->err = msg;
    return s;
}

pwa_status cuda_fail(pwa_ctx *ctx, cudaError_t e, const char *what)
{
    std::string msg = std::string(what) + ": " + cudaGetErrorString(e);
    pwa_status s = (e == cudaErrorMemoryAllocation) ? PWA_ERR_OOM : PWA_ERR_CUDA;
    if (e == cudaErrorMemoryAllocation) cudaGetLastError();   // clear the sticky-free error
    return fail(ctx, s, msg);
}

pwa_status ensure_partials(pwa_ctx *ctx, size_t doubles)
{
    if (doubles <= ctx->partials_cap) return PWA_OK;
    // grows only when the launch shape changes (first evaluation after an upload)
    if (ctx->d_partials) { PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->d_partials); ctx->d_partials = nullptr; }
    ctx->partials_cap = 0;
    PWA_CUDA(ctx, cudaMalloc(&ctx->d_partials, doubles * sizeof(double)));
    ctx->partials_cap = doubles;
    return PWA_OK;
}

pwa_status ensure_scratch(pwa_ctx *ctx, size_t bytes)
{
    if (bytes <= ctx->scratch_cap) return PWA_OK;
    if (ctx->d_scratch) { PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream)); cudaFree(ctx->d_scratch); ctx->d_scratch = nullptr; }
    ctx->scratch_cap = 0;
    PWA_CUDA(ctx, cudaMalloc(&ctx->d_scratch, bytes));
    ctx->scratch_cap = bytes;
    return PWA_OK;
}

static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

static void free_sample(Sample &s)
{
    if (s.amps_owned && s.amps) cudaFree(s.amps);
    if (s.fact_owned) { if (s.mass) cudaFree(s.mass); if (s.ang) cudaFree(s.ang); }
    if (s.weights_owned && s.weights) cudaFree(s.weights);
    s = Sample();
}

// the int8 batched path's per-upload state of the DATA sample (column scales, digit-plane image)
static void drop_i8d(pwa_ctx *ctx)
{
    if (ctx->i8d.planes) cudaFree(ctx->i8d.planes);
    ctx->i8d.planes = nullptr; ctx->i8d.checked = false; ctx->i8d.valid = false;
}

static size_t elem_size(pwa_dtype d) { return d == PWA_F32 ? sizeof(float) : sizeof(double); }

// copy (host or device source) into a fresh device buffer, or borrow a device pointer
static pwa_status take_buffer(pwa_ctx *ctx, const void *src, size_t bytes, uint32_t flags,
                              void **dst, bool *owned)
{
    *dst = nullptr; *owned = false;
    if (bytes == 0) return PWA_OK;
    const bool dev = is_device_ptr(src);
    if (flags & PWA_BORROW) {
        if (!dev) return fail(ctx, PWA_ERR_INVALID_ARG, "PWA_BORROW needs a device pointer");
        if (((uintptr_t)src & 15u) != 0) return fail(ctx, PWA_ERR_INVALID_ARG, "PWA_BORROW pointer must be 16-byte aligned");
        *dst = const_cast<void *>(src);
        return PWA_OK;
    }
    void *buf = nullptr;
    PWA_CUDA(ctx, cudaMalloc(&buf, bytes));
    cudaError_t e = cudaMemcpyAsync(buf, src, bytes, dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { cudaFree(buf); return cuda_fail(ctx, e, "upload copy"); }
    *dst = buf; *owned = true;
    return PWA_OK;
}

static pwa_status check_ready(pwa_ctx *ctx, bool need_M)
{
    if (ctx->data.n_events < 0) return fail(ctx, PWA_ERR_STATE, "no DATA sample uploaded");
    if (need_M && !ctx->M_valid) return fail(ctx, PWA_ERR_STATE, "normalisation matrix missing or stale: call pwa_build_norm");
    return PWA_OK;
}

static bool finite_all(const double *x, size_t k)
{
    for (size_t i = 0; i < k; ++i) if (!isfinite(x[i])) return false;
    return true;
}

static pwa_status unpack_results(pwa_ctx *ctx, int K, double *nll, double *grad, double *parts)
{
    const int n = ctx->n, st = result_stride(n);
    bool nonfinite = false;
    for (int k = 0; k < K; ++k) {
        const double *r = ctx->h_result + (size_t)k * st;
        if (nll) nll[k] = r[0];
        if (parts) { parts[2 * k] = r[1]; parts[2 * k + 1] = r[2]; }
        if (grad) memcpy(grad + (size_t)k * 2 * n, r + 4, sizeof(double) * 2 * n);
        if (r[3] != 0.0 || !finite_all(r, (size_t)st)) nonfinite = true;
    }
    return nonfinite ? PWA_WARN_NONFINITE : PWA_OK;
}

// Waits until the K result records of the most recent enqueue are complete in pinned host memory:
// polls the per-record flags the finishing blocks set (a few microseconds sooner than a stream
// synchronisation: the per-iteration synthesis is latency-bound); every so often it asks the
// stream, so a failed launch is reported instead of spinning forever.
static pwa_status wait_results(pwa_ctx *ctx, int K)
{
    volatile unsigned long long *flags = ctx->h_flags;
    const unsigned long long seq = ctx->seq;
    int k = 0;
    for (unsigned spins = 0;; ++spins) {
        while (k < K && flags[k] == seq) ++k;
        if (k == K) break;
        if ((spins & 1023u) == 1023u) {
            cudaError_t e = cudaStreamQuery(ctx->stream);
            if (e == cudaSuccess) {              // all work done: the flags are visible by now (or a kernel did not run)
                while (k < K && flags[k] == seq) ++k;
                if (k == K) break;
                return fail(ctx, PWA_ERR_CUDA, "evaluation finished without publishing its results");
            }
            if (e != cudaErrorNotReady) return cuda_fail(ctx, e, "waiting for results");
        }
    }
    __sync_synchronize();
    return PWA_OK;
}

// V -> pinned staging h_V.  A previous enqueue may still be copying h_V to the device (cudaMemcpyAsync in
// upload_V): the event recorded behind that copy is waited for first, so back-to-back enqueues with different V
// never race ("V is copied before return", pwa.h).
static pwa_status stage_V(pwa_ctx *ctx, int K, const double *V)
{
    const size_t cnt = (size_t)K * 2 * ctx->n;
    if (!finite_all(V, cnt)) return fail(ctx, PWA_ERR_INVALID_ARG, "V contains non-finite values");
    if (ctx->ev_V_pending) { PWA_CUDA(ctx, cudaEventSynchronize(ctx->ev_V)); ctx->ev_V_pending = false; }
    memcpy(ctx->h_V, V, sizeof(double) * cnt);
    return PWA_OK;
}

// staged h_V -> d_V on the context's stream (only the paths that read V from device memory need it)
static pwa_status upload_V(pwa_ctx *ctx, int K)
{
    PWA_CUDA(ctx, cudaMemcpyAsync(ctx->d_V, ctx->h_V, sizeof(double) * (size_t)K * 2 * ctx->n, cudaMemcpyHostToDevice, ctx->stream));
    PWA_CUDA(ctx, cudaEventRecord(ctx->ev_V, ctx->stream));
    ctx->ev_V_pending = true;
    return PWA_OK;
}

// ---- resident evaluation grid (option "resident", data_term_tma.cu) ------------------------------------------------
// Mailbox words are (tag << 32 | 32 bits of payload), tag = low half of the evaluation's sequence number; tag 0xffffffff
// in every word means quit and is never used for a command.
static const unsigned kResidentQuitTag = 0xffffffffu;

static void mailbox_fill(pwa_ctx *ctx, unsigned tag)
{
    volatile unsigned long long *w = ctx->h_cmd;
    for (int k = 0; k < 4 * kMaxFastWaves; ++k) w[k] = (unsigned long long)tag << 32;
    __sync_synchronize();
}

// Ends the grid (quit command + stream synchronisation).  Called by every entry point that enqueues other work on the
// stream or changes what the grid reads (samples, M, options), so that a resident grid is never in anybody's way.
static pwa_status resident_stop(pwa_ctx *ctx)
{
    if (!ctx->resident_running) return PWA_OK;
    mailbox_fill(ctx, kResidentQuitTag);
    ctx->resident_running = false;
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return PWA_OK;
}

static pwa_status resident_start(pwa_ctx *ctx, bool *started)
{
    if ((unsigned)ctx->seq == kResidentQuitTag) ++ctx->seq;
    mailbox_fill(ctx, (unsigned)ctx->seq);                      // commands carry later numbers
    // the device copy of the mailbox starts with the same tags (staged through h_V: the host may write the first command
    // into h_cmd before the copy has run)
    if (ctx->ev_V_pending) { PWA_CUDA(ctx, cudaEventSynchronize(ctx->ev_V)); ctx->ev_V_pending = false; }
    unsigned long long *stage = reinterpret_cast<unsigned long long *>(ctx->h_V);
    for (int k = 0; k < 4 * ctx->n; ++k) stage[k] = (unsigned long long)(unsigned)ctx->seq << 32;
    PWA_CUDA(ctx, cudaMemcpyAsync(ctx->d_cmd, stage, sizeof(unsigned long long) * 4 * (size_t)ctx->n, cudaMemcpyHostToDevice, ctx->stream));
    PWA_CUDA(ctx, cudaEventRecord(ctx->ev_V, ctx->stream));
    ctx->ev_V_pending = true;
    pwa_status s = launch_resident(ctx, started);
    if (s == PWA_OK && *started) ctx->resident_running = true;
    return s;
}

static void resident_send(pwa_ctx *ctx, const double *V, unsigned tag)
{
    const unsigned *half = reinterpret_cast<const unsigned *>(V);
    volatile unsigned long long *w = ctx->h_cmd;
    const int nw = 4 * ctx->n;
    for (int k = 0; k < nw; ++k) w[k] = ((unsigned long long)tag << 32) | half[k];
    __sync_synchronize();
}

// One evaluation through the mailbox.  The record comes back as 2 (4 + 2n) tagged words in mapped host memory and is
// complete when every word carries this evaluation's tag; it is then unpacked into h_result[0] for unpack_results.
// *done = false: the shape is not served by the resident kernel (the caller evaluates by a launch).
static pwa_status resident_eval(pwa_ctx *ctx, const double *V, bool *done)
{
    *done = false;
    if (!ctx->resident_running) {
        bool started = false;
        pwa_status s = resident_start(ctx, &started);
        if (s != PWA_OK || !started) return s;
    }
    const int nwords = 2 * (4 + 2 * ctx->n);
    volatile unsigned long long *r = ctx->h_rres;
    ctx->last_K = 1;
    for (int restarts = 0;; ++restarts) {
        ++ctx->seq;
        if ((unsigned)ctx->seq == kResidentQuitTag) ++ctx->seq;  // the grid follows any forward jump of the tag
        const unsigned tag = (unsigned)ctx->seq;
        resident_send(ctx, V, tag);
        bool answered = false;
        for (unsigned spins = 0; !answered; ++spins) {
            if ((unsigned)(r[nwords - 1] >> 32) == tag) {
                int k = 0;
                while (k < nwords && (unsigned)(r[k] >> 32) == tag) ++k;
                answered = k == nwords;
                continue;
            }
            if ((spins & 0xfffffu) != 0xfffffu) continue;
            cudaError_t e = cudaStreamQuery(ctx->stream);      // every ~1e6 polls: is the grid still there?
            if (e == cudaSuccess) break;                       // it ended (idle for ~2 s before this command)
            if (e != cudaErrorNotReady) return cuda_fail(ctx, e, "waiting for the resident grid");
            if (spins > (1u << 31)) return fail(ctx, PWA_ERR_CUDA, "resident grid does not answer");
        }
        if (answered) break;
        ctx->resident_running = false;
        if (restarts == 3) return fail(ctx, PWA_ERR_CUDA, "resident grid keeps ending before it answers");
        bool started = false;
        pwa_status s = resident_start(ctx, &started);          // start it again, send the command again under a new number
        if (s != PWA_OK) return s;
        if (!started) return fail(ctx, PWA_ERR_CUDA, "resident grid could not be restarted");
    }
    __sync_synchronize();
    unsigned *dst = reinterpret_cast<unsigned *>(ctx->h_result);
    for (int k = 0; k < nwords; ++k) dst[k] = (unsigned)r[k];
    ctx->h_flags[0] = ctx->seq;                                 // a pwa_fetch(1) behind this call returns the same record
    *done = true;
    return PWA_OK;
}

static pwa_status enqueue_evals(pwa_ctx *ctx, int K, bool batched)
{
    const int n = ctx->n;
    const bool fast = (n == 4 || n == 8 || n == 16 || n == 32 || n == 64) && ctx->opt_data_term != 99;
    const bool need_dV = batched || (!fast && !ctx->data.factored);
    pwa_status s = PWA_OK;
    if (need_dV) { s = upload_V(ctx, K); if (s != PWA_OK) return s; }
    ++ctx->seq;                                  // the finishing blocks publish this id in h_flags[k]
    if (batched) {
        s = launch_batch(ctx, K);
    } else {
        for (int k = 0; k < K && s == PWA_OK; ++k)
            s = launch_data_term(ctx, ctx->h_V + (size_t)k * 2 * n, k, nullptr);
    }
    if (s != PWA_OK) return s;
    ctx->last_K = K;                             // results arrive in h_result by the kernels' own stores (no D2H copy)
    return PWA_OK;
}

}  // namespace pwa

using namespace pwa;

extern "C" {

const char *pwa_status_string(pwa_status s)
{
    switch (s) {
    case PWA_OK: return "PWA_OK";
    case PWA_ERR_INVALID_ARG: return "PWA_ERR_INVALID_ARG";
    case PWA_ERR_STATE: return "PWA_ERR_STATE";
    case PWA_ERR_OOM: return "PWA_ERR_OOM";
    case PWA_ERR_CUDA: return "PWA_ERR_CUDA";
    case PWA_ERR_UNSUPPORTED: return "PWA_ERR_UNSUPPORTED";
    case PWA_WARN_NONFINITE: return "PWA_WARN_NONFINITE";
    }
    return "PWA_?";
}

const char *pwa_last_error(const pwa_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

pwa_status pwa_create(pwa_ctx **out, int32_t n_waves, pwa_dtype storage, int32_t device, void *cuda_stream)
{
    if (!out) return PWA_ERR_INVALID_ARG;
    *out = nullptr;
    if (n_waves < 1 || n_waves > 256) return PWA_ERR_INVALID_ARG;
    if (storage != PWA_F64 && storage != PWA_F32) return PWA_ERR_INVALID_ARG;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) { cudaGetLastError(); return PWA_ERR_CUDA; }
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return PWA_ERR_CUDA; }
    pwa_ctx *ctx = new (std::nothrow) pwa_ctx();
    if (!ctx) return PWA_ERR_OOM;
    ctx->n = n_waves; ctx->storage = storage; ctx->device = device; ctx->stream = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) ctx->sm_count = prop.multiProcessorCount;
    const size_t n = (size_t)n_waves;
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_M, sizeof(double) * 2 * n * n);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_ticket, 4 * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemset(ctx->d_ticket, 0, 4 * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_result, sizeof(double) * kMaxK * result_stride(n_waves));
    if (e == cudaSuccess) e = cudaHostAlloc(&ctx->h_result, sizeof(double) * kMaxK * result_stride(n_waves), cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&ctx->dev_result, ctx->h_result, 0);
    if (e == cudaSuccess) e = cudaHostAlloc(&ctx->h_flags, sizeof(unsigned long long) * kMaxK, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&ctx->dev_flags, ctx->h_flags, 0);
    if (e == cudaSuccess) memset(ctx->h_flags, 0, sizeof(unsigned long long) * kMaxK);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_V, sizeof(double) * kMaxK * 2 * n);
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_V, sizeof(double) * kMaxK * 2 * n);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_V, cudaEventDisableTiming);
    // mailbox of the resident grid (option "resident"): tagged command words, tagged record, device copy {seq, V}
    const size_t cmd_words = 4 * (size_t)kMaxFastWaves, rres_words = 2 * (4 + 2 * (size_t)kMaxFastWaves);
    if (e == cudaSuccess) e = cudaHostAlloc(&ctx->h_cmd, sizeof(unsigned long long) * cmd_words, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&ctx->dev_cmd_host, ctx->h_cmd, 0);
    if (e == cudaSuccess) memset(ctx->h_cmd, 0, sizeof(unsigned long long) * cmd_words);
    if (e == cudaSuccess) e = cudaHostAlloc(&ctx->h_rres, sizeof(unsigned long long) * rres_words, cudaHostAllocMapped);
    if (e == cudaSuccess) e = cudaHostGetDevicePointer(&ctx->dev_rres, ctx->h_rres, 0);
    if (e == cudaSuccess) memset(ctx->h_rres, 0, sizeof(unsigned long long) * rres_words);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_cmd, sizeof(unsigned long long) * cmd_words);
    if (e == cudaSuccess) e = cudaMemset(ctx->d_cmd, 0, sizeof(unsigned long long) * cmd_words);
    // per-block partial slots of every single-V pass (data term: 2 + 2n components, resonance gradient: up to
    // 2 + 4 kMaxRes), sized here for the largest grid any launcher uses (<= 16 blocks per SM), so that no
    // evaluation call ever allocates (pwa.h, general rules)
    if (e == cudaSuccess) {
        const size_t comps = (size_t)(2 + 2 * n_waves > 2 + 4 * kMaxRes ? 2 + 2 * n_waves : 2 + 4 * kMaxRes);
        ctx->partials_cap = comps * (size_t)ctx->sm_count * 16;
        e = cudaMalloc(&ctx->d_partials, ctx->partials_cap * sizeof(double));
        if (e != cudaSuccess) ctx->partials_cap = 0;
    }
    if (e != cudaSuccess) { cudaGetLastError(); pwa_destroy(ctx); return e == cudaErrorMemoryAllocation ? PWA_ERR_OOM : PWA_ERR_CUDA; }
    ctx->h_M.assign(2 * n * n, 0.0);
    *out = ctx;
    return PWA_OK;
}

void pwa_destroy(pwa_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    if (ctx->resident_running && ctx->h_cmd) { mailbox_fill(ctx, kResidentQuitTag); ctx->resident_running = false; }
    cudaStreamSynchronize(ctx->stream);
    free_sample(ctx->data);
    free_sample(ctx->mc);
    drop_i8d(ctx);
    if (ctx->d_M) cudaFree(ctx->d_M);
    if (ctx->d_ticket) cudaFree(ctx->d_ticket);
    if (ctx->d_result) cudaFree(ctx->d_result);
    if (ctx->h_result) cudaFreeHost(ctx->h_result);
    if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
    if (ctx->d_V) cudaFree(ctx->d_V);
    if (ctx->h_V) cudaFreeHost(ctx->h_V);
    if (ctx->ev_V) cudaEventDestroy(ctx->ev_V);
    if (ctx->h_cmd) cudaFreeHost(ctx->h_cmd);
    if (ctx->h_rres) cudaFreeHost(ctx->h_rres);
    if (ctx->d_cmd) cudaFree(ctx->d_cmd);
    if (ctx->d_partials) cudaFree(ctx->d_partials);
    if (ctx->d_scratch) cudaFree(ctx->d_scratch);
    if (ctx->d_H) cudaFree(ctx->d_H);
    cudaGetLastError();
    delete ctx;
}

pwa_status pwa_upload_events(pwa_ctx *ctx, pwa_sample which, const void *amps, int64_t n_events,
                             int64_t n_generated, uint32_t flags)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (which != PWA_DATA && which != PWA_MC) return fail(ctx, PWA_ERR_INVALID_ARG, "bad sample id");
    if (n_events < 0 || (n_events > 0 && !amps)) return fail(ctx, PWA_ERR_INVALID_ARG, "bad amps / n_events");
    if (flags > PWA_BORROW) return fail(ctx, PWA_ERR_INVALID_ARG, "bad flags");
    if (which == PWA_MC && n_generated < n_events) return fail(ctx, PWA_ERR_INVALID_ARG, "n_generated < n_events");
    if (which == PWA_MC && n_generated < 1) return fail(ctx, PWA_ERR_INVALID_ARG, "n_generated must be >= 1");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    void *buf = nullptr; bool owned = false;
    const size_t bytes = (size_t)n_events * (size_t)ctx->n * 2 * elem_size(ctx->storage);
    pwa_status s = take_buffer(ctx, amps, bytes, flags, &buf, &owned);
    if (s != PWA_OK) return s;
    Sample &smp = (which == PWA_DATA) ? ctx->data : ctx->mc;
    free_sample(smp);
    smp.amps = buf; smp.amps_owned = owned; smp.factored = false;
    if (which == PWA_DATA) { ctx->tmap_cache.valid = false; drop_i8d(ctx); }
    smp.n_events = n_events; smp.n_gen = n_generated;
    if (which == PWA_MC) { ctx->M_valid = false; return prepare_norm_i8(ctx); }
    return PWA_OK;
}

pwa_status pwa_upload_events_factored(pwa_ctx *ctx, pwa_sample which, const double *mass, const void *ang,
                                      int32_t n_ang, int64_t n_events, int64_t n_generated, uint32_t flags)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (which != PWA_DATA && which != PWA_MC) return fail(ctx, PWA_ERR_INVALID_ARG, "bad sample id");
    if (n_ang < 1 || n_ang > kMaxAng) return fail(ctx, PWA_ERR_INVALID_ARG, "n_ang must be in [1, 4]");
    if (n_events < 0 || (n_events > 0 && (!mass || !ang))) return fail(ctx, PWA_ERR_INVALID_ARG, "bad mass / ang / n_events");
    if (flags > PWA_BORROW) return fail(ctx, PWA_ERR_INVALID_ARG, "bad flags");
    if (which == PWA_MC && (n_generated < n_events || n_generated < 1)) return fail(ctx, PWA_ERR_INVALID_ARG, "bad n_generated");
    if (ctx->n > kMaxFastWaves) return fail(ctx, PWA_ERR_UNSUPPORTED, "factored mode needs n <= 64");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    void *bm = nullptr, *ba = nullptr; bool om = false, oa = false;
    pwa_status s = take_buffer(ctx, mass, (size_t)n_events * sizeof(double), flags, &bm, &om);
    if (s != PWA_OK) return s;
    s = take_buffer(ctx, ang, (size_t)n_events * (size_t)n_ang * 2 * elem_size(ctx->storage), flags, &ba, &oa);
    if (s != PWA_OK) { if (om) cudaFree(bm); return s; }
    Sample &smp = (which == PWA_DATA) ? ctx->data : ctx->mc;
    free_sample(smp);
    smp.mass = (double *)bm; smp.ang = ba; smp.fact_owned = om || oa; smp.n_ang = n_ang; smp.factored = true;
    smp.n_events = n_events; smp.n_gen = n_generated;
    if (which == PWA_MC) { ctx->M_valid = false; ctx->i8q.valid = false; }
    else drop_i8d(ctx);
    return PWA_OK;
}

pwa_status pwa_set_weights(pwa_ctx *ctx, pwa_sample which, const double *w, uint32_t flags)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (which != PWA_DATA && which != PWA_MC) return fail(ctx, PWA_ERR_INVALID_ARG, "bad sample id");
    if (flags > PWA_BORROW) return fail(ctx, PWA_ERR_INVALID_ARG, "bad flags");
    Sample &smp = (which == PWA_DATA) ? ctx->data : ctx->mc;
    if (smp.n_events < 0) return fail(ctx, PWA_ERR_STATE, "upload the sample before its weights");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    void *buf = nullptr; bool owned = false;
    if (w != nullptr && smp.n_events > 0) {
        pwa_status s = take_buffer(ctx, w, (size_t)smp.n_events * sizeof(double), flags, &buf, &owned);
        if (s != PWA_OK) return s;
    }
    // sum of the weights = N_data of the eq. 2 form (compensated, index order): found once here, on the host
    double sum_w = 0.0;
    if (buf != nullptr) {
        const size_t cnt = (size_t)smp.n_events;
        std::vector<double> tmp;
        const double *hw = w;
        if (is_device_ptr(w)) {
            tmp.resize(cnt);
            cudaError_t e = cudaMemcpy(tmp.data(), buf, cnt * sizeof(double), cudaMemcpyDeviceToHost);
            if (e != cudaSuccess) { if (owned) cudaFree(buf); return cuda_fail(ctx, e, "reading the weights back"); }
            hw = tmp.data();
        }
        double s = 0.0, c = 0.0;                     // Neumaier
        for (size_t i = 0; i < cnt; ++i) {
            const double x = hw[i], t = s + x;
            c += (fabs(s) >= fabs(x)) ? (s - t) + x : (x - t) + s;
            s = t;
        }
        sum_w = s + c;
        if (!isfinite(sum_w)) { if (owned) cudaFree(buf); return fail(ctx, PWA_ERR_INVALID_ARG, "weights contain non-finite values"); }
    }
    if (smp.weights_owned && smp.weights) cudaFree(smp.weights);
    smp.weights = (double *)buf; smp.weights_owned = owned; smp.sum_w = sum_w;
    if (which == PWA_MC) ctx->M_valid = false;
    return PWA_OK;
}

pwa_status pwa_set_wave_map(pwa_ctx *ctx, int32_t n_res, const int32_t *res_of_wave, const int32_t *ang_of_wave)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (n_res < 1 || n_res > kMaxRes || !res_of_wave || !ang_of_wave) return fail(ctx, PWA_ERR_INVALID_ARG, "bad wave map");
    if (ctx->n > kMaxFastWaves) return fail(ctx, PWA_ERR_UNSUPPORTED, "factored mode needs n <= 64");
    std::vector<int32_t> pair(n_res * kMaxAng, -1);
    for (int a = 0; a < ctx->n; ++a) {
        if (res_of_wave[a] < 0 || res_of_wave[a] >= n_res || ang_of_wave[a] < 0 || ang_of_wave[a] >= kMaxAng)
            return fail(ctx, PWA_ERR_INVALID_ARG, "wave map entry out of range");
        int32_t &slot = pair[res_of_wave[a] * kMaxAng + ang_of_wave[a]];
        if (slot >= 0) return fail(ctx, PWA_ERR_INVALID_ARG, "two waves share one (resonance, angular structure) pair");
        slot = a;
    }
    ctx->n_res = n_res;
    ctx->res_of_wave.assign(res_of_wave, res_of_wave + ctx->n);
    ctx->ang_of_wave.assign(ang_of_wave, ang_of_wave + ctx->n);
    ctx->wave_of_pair = pair;
    ctx->res_set = false;
    ctx->M_valid = false;
    return PWA_OK;
}

pwa_status pwa_set_resonances(pwa_ctx *ctx, const double *mass0, const double *width0)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (ctx->n_res < 1) return fail(ctx, PWA_ERR_STATE, "pwa_set_wave_map not called");
    if (!mass0 || !width0 || !finite_all(mass0, ctx->n_res) || !finite_all(width0, ctx->n_res))
        return fail(ctx, PWA_ERR_INVALID_ARG, "bad resonance parameters");
    ctx->mass0.assign(mass0, mass0 + ctx->n_res);
    ctx->width0.assign(width0, width0 + ctx->n_res);
    ctx->res_set = true;
    if (ctx->mc.factored) ctx->M_valid = false;
    return PWA_OK;
}

pwa_status pwa_build_norm(pwa_ctx *ctx, double *M_out)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (ctx->mc.n_events < 0) return fail(ctx, PWA_ERR_STATE, "no MC sample uploaded");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    pwa_status s = launch_norm_build(ctx);
    if (s != PWA_OK) return s;
    ctx->M_valid = true;
    if (M_out) {
        const size_t cnt = 2 * (size_t)ctx->n * ctx->n;
        PWA_CUDA(ctx, cudaMemcpyAsync(ctx->h_M.data(), ctx->d_M, sizeof(double) * cnt, cudaMemcpyDeviceToHost, ctx->stream));
        PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        memcpy(M_out, ctx->h_M.data(), sizeof(double) * cnt);
    }
    return PWA_OK;
}

pwa_status pwa_norm_error_bound(pwa_ctx *ctx, double *bound, int32_t *which_path)
{
    if (!ctx || !bound) return PWA_ERR_INVALID_ARG;
    if (!ctx->M_valid) return fail(ctx, PWA_ERR_STATE, "normalisation matrix missing or stale: call pwa_build_norm");
    *bound = (ctx->M_path == 1 || ctx->M_path == 3) ? norm_i8_error_bound(ctx) : 0.0;
    if (which_path) *which_path = ctx->M_path;
    return PWA_OK;
}

pwa_status pwa_batch_path(pwa_ctx *ctx, int32_t *which_path, double *err_rel)
{
    if (!ctx || !which_path) return PWA_ERR_INVALID_ARG;
    if (ctx->batch_path < 0) return fail(ctx, PWA_ERR_STATE, "no batched evaluation yet");
    *which_path = ctx->batch_path;
    if (err_rel) *err_rel = ctx->batch_path == 2 ? batch_i8_error_estimate(ctx) : 0.0;
    return PWA_OK;
}

pwa_status pwa_set_norm(pwa_ctx *ctx, const double *M)
{
    if (!ctx || !M) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    const size_t cnt = 2 * (size_t)ctx->n * ctx->n;
    if (!finite_all(M, cnt)) return fail(ctx, PWA_ERR_INVALID_ARG, "M contains non-finite values");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(ctx->h_M.data(), M, sizeof(double) * cnt);
    PWA_CUDA(ctx, cudaMemcpyAsync(ctx->d_M, ctx->h_M.data(), sizeof(double) * cnt, cudaMemcpyHostToDevice, ctx->stream));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->M_valid = true;
    ctx->M_path = 0;
    return PWA_OK;
}

pwa_status pwa_nll_grad_enqueue(pwa_ctx *ctx, const double *V)
{
    if (!ctx || !V) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    pwa_status s = check_ready(ctx, true);
    if (s != PWA_OK) return s;
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    s = stage_V(ctx, 1, V);
    if (s != PWA_OK) return s;
    return enqueue_evals(ctx, 1, false);
}

pwa_status pwa_nll_grad_batch_enqueue(pwa_ctx *ctx, int32_t K, const double *V)
{
    if (!ctx || !V) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (K < 1 || K > kMaxK) return fail(ctx, PWA_ERR_INVALID_ARG, "K must be in [1, 1024]");
    pwa_status s = check_ready(ctx, true);
    if (s != PWA_OK) return s;
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    s = stage_V(ctx, K, V);
    if (s != PWA_OK) return s;
    return enqueue_evals(ctx, K, true);
}

pwa_status pwa_fetch(pwa_ctx *ctx, int32_t K, double *nll, double *grad, double *parts)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    if (K < 1 || K != ctx->last_K) return fail(ctx, PWA_ERR_STATE, "pwa_fetch: K does not match the last enqueue");
    pwa_status s = wait_results(ctx, K);
    if (s != PWA_OK) return s;
    return unpack_results(ctx, K, nll, grad, parts);
}

pwa_status pwa_nll_grad(pwa_ctx *ctx, const double *V, double *nll, double *grad, double *parts)
{
    if (!ctx || !V || !nll || !grad) return ctx ? fail(ctx, PWA_ERR_INVALID_ARG, "null argument") : PWA_ERR_INVALID_ARG;
    if (ctx->opt_resident) {                         // evaluation through the resident grid's mailbox: no launch
        pwa_status s = check_ready(ctx, true);
        if (s != PWA_OK) return s;
        if (!finite_all(V, 2 * (size_t)ctx->n)) return fail(ctx, PWA_ERR_INVALID_ARG, "V contains non-finite values");
        PWA_CUDA(ctx, cudaSetDevice(ctx->device));
        bool done = false;
        s = resident_eval(ctx, V, &done);
        if (s != PWA_OK) return s;
        if (done) return unpack_results(ctx, 1, nll, grad, parts);
    }
    pwa_status s = pwa_nll_grad_enqueue(ctx, V);
    if (s != PWA_OK) return s;
    return pwa_fetch(ctx, 1, nll, grad, parts);
}

pwa_status pwa_nll_grad_batch(pwa_ctx *ctx, int32_t K, const double *V, double *nll, double *grad, double *parts)
{
    if (!ctx || !V || !nll || !grad) return ctx ? fail(ctx, PWA_ERR_INVALID_ARG, "null argument") : PWA_ERR_INVALID_ARG;
    pwa_status s = pwa_nll_grad_batch_enqueue(ctx, K, V);
    if (s != PWA_OK) return s;
    return pwa_fetch(ctx, K, nll, grad, parts);
}

pwa_status pwa_data_term_enqueue(pwa_ctx *ctx, const double *V, double *out_dev)
{
    if (!ctx || !V || !out_dev) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    pwa_status s = check_ready(ctx, false);
    if (s != PWA_OK) return s;
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    s = stage_V(ctx, 1, V);
    if (s != PWA_OK) return s;
    const int n = ctx->n;
    const bool fast = (n == 4 || n == 8 || n == 16 || n == 32 || n == 64) && ctx->opt_data_term != 99;
    if (!fast && !ctx->data.factored) { s = upload_V(ctx, 1); if (s != PWA_OK) return s; }
    ctx->last_K = 0;                             // no result record is written: a later pwa_fetch must not return a stale one
    return launch_data_term(ctx, ctx->h_V, 0, out_dev);
}

pwa_status pwa_assemble_host(int32_t n, double L_data, const double *T, const double *M, const double *V,
                             double *nll, double *grad, double *parts)
{
    if (n < 1 || !T || !M || !V || !nll || !grad) return PWA_ERR_INVALID_ARG;
    double norm = 0.0;
    for (int a = 0; a < n; ++a) {
        double mr = 0.0, mi = 0.0;
        for (int b = 0; b < n; ++b) {
            const double Mr = M[((size_t)a * n + b) * 2], Mi = M[((size_t)a * n + b) * 2 + 1];
            mr += Mr * V[2 * b] - Mi * V[2 * b + 1];
            mi += Mr * V[2 * b + 1] + Mi * V[2 * b];
        }
        norm += V[2 * a] * mr + V[2 * a + 1] * mi;
        grad[2 * a] = -2.0 * T[2 * a] + 2.0 * mr;
        grad[2 * a + 1] = 2.0 * T[2 * a + 1] + 2.0 * mi;
    }
    *nll = -(L_data - norm);
    if (parts) { parts[0] = L_data; parts[1] = norm; }
    return PWA_OK;
}

pwa_status pwa_assemble_host_shards(int32_t n, int32_t R, const double *terms, const double *M, const double *V,
                                    int32_t likelihood, double n_data, double *nll, double *grad, double *parts)
{
    if (n < 1 || R < 1 || !terms || !M || !V || !nll || !grad || (likelihood != 0 && likelihood != 1)) return PWA_ERR_INVALID_ARG;
    const int NC = 2 + 2 * n;
    std::vector<double> tot(terms, terms + NC);
    for (int r = 1; r < R; ++r)                                     // shard order: the same bits on every rank
        for (int c = 0; c < NC; ++c) tot[c] += terms[(size_t)r * NC + c];
    pwa_status s = likelihood == 1 ? pwa_assemble_host_eq2(n, n_data, tot[0], tot.data() + 2, M, V, nll, grad, parts)
                                   : pwa_assemble_host(n, tot[0], tot.data() + 2, M, V, nll, grad, parts);
    if (s != PWA_OK) return s;
    return (tot[1] != 0.0 || !finite_all(tot.data(), (size_t)NC)) ? PWA_WARN_NONFINITE : PWA_OK;
}

pwa_status pwa_norm_sums(pwa_ctx *ctx, double *G_out, int64_t *n_gen_out)
{
    if (!ctx || !G_out || !n_gen_out) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (ctx->mc.n_events < 0) return fail(ctx, PWA_ERR_STATE, "no MC sample uploaded");
    if (!ctx->M_valid) return fail(ctx, PWA_ERR_STATE, "normalisation matrix missing or stale: call pwa_build_norm");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t cnt = 2 * (size_t)ctx->n * ctx->n;
    PWA_CUDA(ctx, cudaMemcpyAsync(ctx->h_M.data(), ctx->d_M, sizeof(double) * cnt, cudaMemcpyDeviceToHost, ctx->stream));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const double ng = (double)ctx->mc.n_gen;
    for (size_t t = 0; t < cnt; ++t) G_out[t] = ctx->h_M[t] * ng;
    *n_gen_out = ctx->mc.n_gen;
    return PWA_OK;
}

pwa_status pwa_combine_norm_host(int32_t n, int32_t R, const double *G, const int64_t *n_gen, double *M_out,
                                 int64_t *n_gen_total)
{
    if (n < 1 || R < 1 || !G || !n_gen || !M_out) return PWA_ERR_INVALID_ARG;
    const size_t cnt = 2 * (size_t)n * n;
    int64_t ng = 0;
    for (int r = 0; r < R; ++r) { if (n_gen[r] < 0) return PWA_ERR_INVALID_ARG; ng += n_gen[r]; }
    if (ng < 1) return PWA_ERR_INVALID_ARG;
    for (size_t t = 0; t < cnt; ++t) M_out[t] = G[t];
    for (int r = 1; r < R; ++r)                                     // shard order: the same bits on every rank
        for (size_t t = 0; t < cnt; ++t) M_out[t] += G[(size_t)r * cnt + t];
    const double den = (double)ng;
    for (size_t t = 0; t < cnt; ++t) M_out[t] /= den;
    if (n_gen_total) *n_gen_total = ng;
    return PWA_OK;
}

pwa_status pwa_fumili_hessian(pwa_ctx *ctx, const double *V, double *H, int32_t with_norm)
{
    if (!ctx || !V || !H) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    pwa_status s = check_ready(ctx, with_norm != 0);
    if (s != PWA_OK) return s;
    if (ctx->data.factored && !ctx->res_set) return fail(ctx, PWA_ERR_STATE, "pwa_set_resonances not called");
    if (ctx->data.weights) return fail(ctx, PWA_ERR_UNSUPPORTED, "pwa_fumili_hessian does not take event weights");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    s = stage_V(ctx, 1, V);
    if (s != PWA_OK) return s;
    const size_t n = (size_t)ctx->n, cnt = 4 * n * n;
    if (ctx->data.n_events == 0) { memset(H, 0, sizeof(double) * cnt); return PWA_OK; }
    s = upload_V(ctx, 1);
    if (s != PWA_OK) return s;
    // H goes through the tail of the M-partials scratch is NOT safe (the Gram kernel owns it): own buffer
    if (!ctx->d_H) PWA_CUDA(ctx, cudaMalloc(&ctx->d_H, sizeof(double) * cnt));
    s = launch_fumili(ctx, ctx->d_H, with_norm != 0);
    if (s != PWA_OK) return s;
    PWA_CUDA(ctx, cudaMemcpyAsync(H, ctx->d_H, sizeof(double) * cnt, cudaMemcpyDeviceToHost, ctx->stream));
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return finite_all(H, cnt) ? PWA_OK : PWA_WARN_NONFINITE;
}

pwa_status pwa_assemble_host_eq2(int32_t n, double n_data, double L_data, const double *T, const double *M,
                                 const double *V, double *nll, double *grad, double *parts)
{
    if (n < 1 || !(n_data > 0.0) || !T || !M || !V || !nll || !grad) return PWA_ERR_INVALID_ARG;
    double norm = 0.0;
    for (int a = 0; a < n; ++a) {
        double mr = 0.0, mi = 0.0;
        for (int b = 0; b < n; ++b) {
            const double Mr = M[((size_t)a * n + b) * 2], Mi = M[((size_t)a * n + b) * 2 + 1];
            mr += Mr * V[2 * b] - Mi * V[2 * b + 1];
            mi += Mr * V[2 * b + 1] + Mi * V[2 * b];
        }
        norm += V[2 * a] * mr + V[2 * a + 1] * mi;
        grad[2 * a] = mr;  grad[2 * a + 1] = mi;                   // (M V)_a for now
    }
    const double gw = 2.0 * (n_data / norm);
    for (int a = 0; a < n; ++a) {
        grad[2 * a] = -2.0 * T[2 * a] + gw * grad[2 * a];
        grad[2 * a + 1] = 2.0 * T[2 * a + 1] + gw * grad[2 * a + 1];
    }
    *nll = -L_data + n_data * log(norm);
    if (parts) { parts[0] = L_data; parts[1] = norm; }
    return PWA_OK;
}

pwa_status pwa_grad_to_polar(int32_t n, const double *V, const double *grad, double *grad_polar)
{
    if (n < 1 || !V || !grad || !grad_polar) return PWA_ERR_INVALID_ARG;
    for (int a = 0; a < n; ++a) {
        const double x = V[2 * a], y = V[2 * a + 1], r = sqrt(x * x + y * y);
        const double gx = grad[2 * a], gy = grad[2 * a + 1];
        grad_polar[2 * a] = r > 0.0 ? (gx * x + gy * y) / r : gx;   // d/dr = gx cos(phi) + gy sin(phi); phi := 0 at r = 0
        grad_polar[2 * a + 1] = -y * gx + x * gy;                    // d/dphi
    }
    return PWA_OK;
}

pwa_status pwa_fix_phase_host(int32_t n, int32_t ref, double *V, double *grad)
{
    if (n < 1 || ref < 0 || ref >= n || !V) return PWA_ERR_INVALID_ARG;
    const double xr = V[2 * ref], yr = V[2 * ref + 1], r = hypot(xr, yr);
    if (r > 0.0) {
        const double c = xr / r, s = -yr / r;                       // exp(-i arg V_ref) = conj(V_ref) / |V_ref|
        for (int a = 0; a < n; ++a) {
            const double x = V[2 * a], y = V[2 * a + 1];
            V[2 * a] = x * c - y * s; V[2 * a + 1] = x * s + y * c;
            if (grad) {
                const double gx = grad[2 * a], gy = grad[2 * a + 1];
                grad[2 * a] = gx * c - gy * s; grad[2 * a + 1] = gx * s + gy * c;
            }
        }
        V[2 * ref] = r;
    }
    V[2 * ref + 1] = 0.0;
    if (grad) grad[2 * ref + 1] = 0.0;
    return PWA_OK;
}

pwa_status pwa_polar_to_cartesian(int32_t n, const double *r_phi, double *V)
{
    if (n < 1 || !r_phi || !V) return PWA_ERR_INVALID_ARG;
    for (int a = 0; a < n; ++a) {
        V[2 * a] = r_phi[2 * a] * cos(r_phi[2 * a + 1]);
        V[2 * a + 1] = r_phi[2 * a] * sin(r_phi[2 * a + 1]);
    }
    return PWA_OK;
}

pwa_status pwa_res_grad(pwa_ctx *ctx, const double *V, double *dM, double *dG)
{
    if (!ctx || !V || !dM || !dG) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (ctx->data.n_events < 0 || ctx->mc.n_events < 0) return fail(ctx, PWA_ERR_STATE, "DATA and MC must be uploaded");
    if (!ctx->data.factored || !ctx->mc.factored) return fail(ctx, PWA_ERR_STATE, "pwa_res_grad needs factored uploads");
    if (!finite_all(V, 2 * (size_t)ctx->n)) return fail(ctx, PWA_ERR_INVALID_ARG, "V contains non-finite values");
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    return launch_res_grad(ctx, V, dM, dG);
}

pwa_status pwa_nll_grad_floating(pwa_ctx *ctx, const double *V, const double *mass0, const double *width0, double *nll,
                                 double *grad, double *dnll_dmass, double *dnll_dwidth, double *parts)
{
    if (!ctx || !V || !mass0 || !width0 || !nll || !grad || !dnll_dmass || !dnll_dwidth)
        return ctx ? fail(ctx, PWA_ERR_INVALID_ARG, "null argument") : PWA_ERR_INVALID_ARG;
    if (ctx->data.n_events < 0 || ctx->mc.n_events < 0) return fail(ctx, PWA_ERR_STATE, "DATA and MC must be uploaded");
    if (!ctx->data.factored || !ctx->mc.factored) return fail(ctx, PWA_ERR_STATE, "pwa_nll_grad_floating needs factored uploads");
    if (ctx->data.weights || ctx->mc.weights) return fail(ctx, PWA_ERR_UNSUPPORTED, "event weights are not supported with factored uploads");
    const int n = ctx->n;
    if (!finite_all(V, 2 * (size_t)n)) return fail(ctx, PWA_ERR_INVALID_ARG, "V contains non-finite values");
    pwa_status s = pwa_set_resonances(ctx, mass0, width0);      // M (if any) no longer belongs to these parameters: marked stale
    if (s != PWA_OK) return s;
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    int NC = 0;
    s = launch_floating_passes(ctx, V, &NC);
    if (s != PWA_OK) return s;
    s = wait_results(ctx, 2);
    if (s != PWA_OK) return s;
    // synthesis on the host (a few hundred flops): record 0 = MC pass, record 1 = data pass
    const double *mc = ctx->h_result, *dt = ctx->h_result + NC;
    const int n_res = ctx->n_res, n_ang = ctx->data.n_ang;
    const double inv_ngen = 1.0 / (double)ctx->mc.n_gen;
    const double norm = mc[0] * inv_ngen, L = dt[0];
    const double wN = ctx->opt_likelihood == 1 ? eq2_n_data(ctx) / norm : 1.0;      // eq. 2: the Norm part carries N_data / Norm
    *nll = ctx->opt_likelihood == 1 ? (-L + eq2_n_data(ctx) * log(norm)) : -(L - norm);
    if (parts) { parts[0] = L; parts[1] = norm; }
    for (int a = 0; a < n; ++a) {
        // grad(L_data) = 2 conj(T);  grad(Norm) = 2 M V = (2 / N_gen) conj(T'),  T' = sum_j A_ja conj(S_j)
        grad[2 * a]     = -2.0 * dt[2 + 2 * a] + wN * 2.0 * inv_ngen * mc[2 + 2 * a];
        grad[2 * a + 1] =  2.0 * dt[3 + 2 * a] - wN * 2.0 * inv_ngen * mc[3 + 2 * a];
    }
    for (int r = 0; r < n_res; ++r) {
        double ud[2] = {0.0, 0.0}, um[2] = {0.0, 0.0};              // U_r = sum_s C[r][s] Q2[r][s], C[r][s] = V of wave (r, s)
        for (int sg = 0; sg < n_ang; ++sg) {
            const int w = ctx->wave_of_pair[r * kMaxAng + sg];
            if (w < 0) continue;
            const double cr = V[2 * w], ci = V[2 * w + 1];
            const double *qd = dt + 2 + 2 * (n + r * n_ang + sg), *qm = mc + 2 + 2 * (n + r * n_ang + sg);
            ud[0] += cr * qd[0] - ci * qd[1]; ud[1] += cr * qd[1] + ci * qd[0];
            um[0] += cr * qm[0] - ci * qm[1]; um[1] += cr * qm[1] + ci * qm[0];
        }
        const double Mr = mass0[r], Gr = width0[r];
        // Re( -(2M - iG) U ) = -(2M Ur + G Ui);  Re( iM U ) = -M Ui                      (reading A9, C3)
        const double dL_dM = 2.0 * (-(2.0 * Mr * ud[0] + Gr * ud[1])), dL_dG = 2.0 * (-Mr * ud[1]);
        const double dN_dM = 2.0 * inv_ngen * (-(2.0 * Mr * um[0] + Gr * um[1])), dN_dG = 2.0 * inv_ngen * (-Mr * um[1]);
        dnll_dmass[r] = -dL_dM + wN * dN_dM;
        dnll_dwidth[r] = -dL_dG + wN * dN_dG;
    }
    const bool nonfinite = mc[1] != 0.0 || dt[1] != 0.0 || !isfinite(*nll) || !finite_all(grad, 2 * (size_t)n);
    return nonfinite ? PWA_WARN_NONFINITE : PWA_OK;
}

uint64_t pwa_launch_count(const pwa_ctx *ctx) { return ctx ? ctx->launches : 0; }

int32_t pwa_n_waves(const pwa_ctx *ctx) { return ctx ? ctx->n : 0; }

int32_t pwa_n_res(const pwa_ctx *ctx) { return ctx ? ctx->n_res : 0; }

int64_t pwa_n_events(const pwa_ctx *ctx, pwa_sample which)
{
    if (!ctx || (which != PWA_DATA && which != PWA_MC)) return -1;
    return which == PWA_DATA ? ctx->data.n_events : ctx->mc.n_events;
}

pwa_dtype pwa_storage(const pwa_ctx *ctx) { return ctx ? ctx->storage : PWA_F64; }

pwa_status pwa_sync(pwa_ctx *ctx)
{
    if (!ctx) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    PWA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return PWA_OK;
}

pwa_status pwa_set_option(pwa_ctx *ctx, const char *key, int32_t value)
{
    if (!ctx || !key) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    if (!strcmp(key, "data_term")) ctx->opt_data_term = value;
    else if (!strcmp(key, "norm")) ctx->opt_norm = value;
    else if (!strcmp(key, "batch")) ctx->opt_batch = value;
    else if (!strcmp(key, "l2_resident_mb")) { if (value < -1 || value > 120) return fail(ctx, PWA_ERR_INVALID_ARG, "l2_resident_mb must be in [-1, 120]"); ctx->opt_l2_resident_mb = value; }
    else if (!strcmp(key, "resident")) { if (value != 0 && value != 1) return fail(ctx, PWA_ERR_INVALID_ARG, "resident must be 0 or 1"); ctx->opt_resident = value != 0; }
    else if (!strcmp(key, "likelihood")) { if (value != 0 && value != 1) return fail(ctx, PWA_ERR_INVALID_ARG, "likelihood must be 0 (eq. 3) or 1 (eq. 2)"); ctx->opt_likelihood = value; }
    else if (!strcmp(key, "fix_phase")) { if (value < 0 || value > ctx->n) return fail(ctx, PWA_ERR_INVALID_ARG, "fix_phase must be 0 (off) or a wave number 1 .. n"); ctx->opt_fix_phase = value; }
    else return fail(ctx, PWA_ERR_INVALID_ARG, "unknown option key");
    return PWA_OK;
}

pwa_status pwa_get_option(pwa_ctx *ctx, const char *key, int32_t *value)
{
    if (!ctx || !key || !value) return PWA_ERR_INVALID_ARG;
    if (!strcmp(key, "data_term")) *value = ctx->opt_data_term;
    else if (!strcmp(key, "norm")) *value = ctx->opt_norm;
    else if (!strcmp(key, "batch")) *value = ctx->opt_batch;
    else if (!strcmp(key, "l2_resident_mb")) *value = ctx->opt_l2_resident_mb;
    else if (!strcmp(key, "resident")) *value = ctx->opt_resident ? 1 : 0;
    else if (!strcmp(key, "likelihood")) *value = ctx->opt_likelihood;
    else if (!strcmp(key, "fix_phase")) *value = ctx->opt_fix_phase;
    else return fail(ctx, PWA_ERR_INVALID_ARG, "unknown option key");
    return PWA_OK;
}

pwa_status pwa_microbench(pwa_ctx *ctx, int32_t which, int64_t bytes, double *result)
{
    if (!ctx || !result) return PWA_ERR_INVALID_ARG;
    { pwa_status rs__ = resident_stop(ctx); if (rs__ != PWA_OK) return rs__; }
    PWA_CUDA(ctx, cudaSetDevice(ctx->device));
    return run_microbench(ctx, which, bytes, result);
}

}  // extern "C"
