// noit_resolve_ring.cu -- staged resolve kernel (placeholder: not taken yet).
#include "noit_resolve_common.cuh"

noit_status noit_launch_resolve_ring(noit_ctx* ctx, const ResolveArgs& A, int color_fmt,
                                     cudaStream_t st, bool* taken)
{
    (void)ctx; (void)A; (void)color_fmt; (void)st;
    *taken = false;
    return NOIT_OK;
}
