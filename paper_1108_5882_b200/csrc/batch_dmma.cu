// batch_dmma.cu — tensor-core path of step A8 (placeholder until the DMMA kernel lands).
#include "pwa_internal.h"

namespace pwa {

pwa_status launch_batch_dmma(pwa_ctx *ctx, int K, bool *handled)
{
    (void)ctx; (void)K;
    *handled = false;
    return PWA_OK;
}

}  // namespace pwa
