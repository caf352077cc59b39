// placeholder: replaced by the tcgen05 kernel
#include "kairos_internal.h"
namespace kairos {
int umma_chunk_tile_tokens() { return 4; }
int umma_resident_ctas(const kairos_ctx* ctx) { return ctx->sm_count; }
int umma_init(kairos_ctx*) { return KAIROS_OK; }
int launch_attn_umma(kairos_ctx*, const StepArgs&, const WorkItem*, int32_t, const CombineItem*, int32_t, cudaStream_t, int*) {
    return fail(KAIROS_ERR_UNSUPPORTED, "tcgen05 path not built yet");
}
}
