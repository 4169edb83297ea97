// gs_resident.cu -- the RESIDENT plan (one persistent CTA per environment).  Placeholder: not built yet,
// every model runs the streaming plan.
#include "gs_internal.h"

namespace gs {
size_t resident_blob_bytes(const gs_model_desc *) { return 0; }
int resident_prepare(gs_model *m, const gs_model_desc *desc, void *, size_t, cudaStream_t) {
    if (desc->plan == GS_PLAN_RESIDENT) { set_error("the resident plan is not available in this build"); return GS_EINVAL; }
    m->plan = GS_PLAN_STREAMING;
    return GS_OK;
}
int resident_rollout(gs_model *, gs_tape *, cudaStream_t) { set_error("resident plan unavailable"); return GS_ESTATE; }
int resident_rollout_backward(gs_model *, gs_tape *, int, int, const float *, cudaStream_t) { set_error("resident plan unavailable"); return GS_ESTATE; }
}  // namespace gs
