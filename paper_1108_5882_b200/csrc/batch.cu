// batch.cu — step A8: K starting points evaluated against the same data ("the fits are
// usually repeated with various sets of starting parameters").
// Variant 0 (this file, reference path): K passes of the single-V streaming kernel.
// Variant 1 (batch_dmma.cu): one pass, chained FP64 tensor-core GEMMs
//     S = A V (N x n by n x K),  l += ln|S|^2, R = 1/S,  T = A^T R (n x N by N x K).
// Variant 2 (batch_i8.cu): the same chain as error-free int8 contractions on tcgen05 (fp32 storage, n = 64).
#include "pwa_internal.h"

namespace pwa {

pwa_status launch_batch_dmma(pwa_ctx *ctx, int K, bool *handled);   // batch_dmma.cu

pwa_status launch_batch(pwa_ctx *ctx, int K)
{
    if (ctx->opt_batch != 99 && ctx->data.weights == nullptr) {      // weighted samples: K passes of the weighted streaming kernel
        bool handled = false;
        pwa_status s = launch_batch_i8(ctx, K, &handled);           // fp32 storage, n = 64: int8 tensor cores (batch_i8.cu)
        if (s != PWA_OK) return s;
        if (handled) { ctx->batch_path = 2; return PWA_OK; }
        s = launch_batch_dmma(ctx, K, &handled);
        if (s != PWA_OK) return s;
        if (handled) { ctx->batch_path = 1; return PWA_OK; }
    }
    ctx->batch_path = 0;
    const int n = ctx->n;
    for (int k = 0; k < K; ++k) {
        pwa_status s = launch_data_term(ctx, ctx->h_V + (size_t)k * 2 * n, k, nullptr);
        if (s != PWA_OK) return s;
    }
    return PWA_OK;
}

}  // namespace pwa
