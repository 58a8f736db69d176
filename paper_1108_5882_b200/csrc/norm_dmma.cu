// norm_dmma.cu — tensor-core path of step A6 (placeholder until the DMMA kernel lands).
#include "pwa_internal.h"

namespace pwa {

pwa_status launch_norm_dmma(pwa_ctx *ctx, bool *handled)
{
    (void)ctx;
    *handled = false;
    return PWA_OK;
}

}  // namespace pwa
