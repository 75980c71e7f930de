// sw_sparse_attn_prefill, sm_100a fast path (tcgen05 + TMEM + TMA).  Placeholder until the
// kernel lands: every shape is routed to the generic mma.sync path.
#include "common.cuh"

namespace sw {

bool attn_prefill_sm100_supported(const AttnPrefillArgs&) { return false; }

int32_t launch_attn_prefill_sm100(const AttnPrefillArgs&, cudaStream_t) {
  return fail(SW_ERR_UNSUPPORTED, "sm100 prefill path not built");
}

}  // namespace sw
