// sa_prefill_tc5.cu -- prefill-chunk attention on tcgen05 / TMEM / TMA.
// Placeholder until the kernel lands: the planner asks tc5_supported() and routes prefill
// chunks to the mma.sync kernel while this returns false.
#include "sa_internal.h"

namespace sa {

int32_t tc5_init(sa_kv_pool *pool) {
    pool->tc5_ready = false;
    return SA_OK;
}

bool tc5_supported(const sa_kv_pool *pool) { return pool->tc5_ready; }

cudaError_t launch_prefill_tc5(const sa_kv_pool *, const ReqMeta *, const AttnPlan &, int64_t, const void *, void *,
                               float *, float, cudaStream_t, int32_t *) {
    return cudaErrorNotSupported;
}

}  // namespace sa
