// a5 placeholder until the tcgen05 fused LM-head kernels land (next commit).
#include "awr_common.cuh"
extern "C" {
__attribute__((visibility("default")))
int awr_loss_fwd_bwd_fused_head(const awr_head_batch*, const awr_params*, const awr_head_outputs*,
                                void*, size_t, void*) { return AWR_ERR_PARAM; }
__attribute__((visibility("default")))
size_t awr_head_workspace_bytes(int64_t, int64_t, int64_t, int32_t, int32_t, int32_t) { return 0; }
}
