// kernels_march.cu -- register-marching separable sweep (placeholder until the first GPU validation of
// the gather path).
#include "tslb_internal.h"

bool tslb_march_supported(const tslb_ctx *, const char **why)
{
    if (why) *why = "march kernel not built in this revision";
    return false;
}

cudaError_t tslb_launch_march(tslb_ctx *, cudaStream_t) { return cudaErrorNotSupported; }
