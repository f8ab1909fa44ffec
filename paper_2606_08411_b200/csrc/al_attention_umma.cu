// placeholder until the tcgen05 kernel lands (next commit): everything routes to the plain-ALU kernel
#include "al_internal.h"
bool al_attention_umma_supported(const al_attn_shape*) { return false; }
size_t al_attention_umma_workspace_bytes(const al_handle*, const al_attn_shape*, int, int, int) { return 0; }
al_status al_launch_attention_umma(const al_handle*, const al_attn_shape*, float, const void*, const void*,
                                   const void*, const void*, const void*, const al_lane_desc*, int, int, int,
                                   void*, float*, void*, size_t, cudaStream_t) {
  AL_FAIL(AL_ERR_UNSUPPORTED, "tcgen05 attention kernel not built");
}
