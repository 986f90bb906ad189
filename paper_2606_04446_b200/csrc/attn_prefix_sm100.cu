// Stage (c) prefix pass on tcgen05 / TMEM / TMA (sm_100a).  Placeholder until the kernel lands:
// reports "unsupported" so that the planner routes every shape to the mma.sync path.
#include "common.cuh"

namespace d2sd {

bool attn_prefix_tc_supported(const AttnPlan&) { return false; }

int32_t launch_attn_prefix_tc(const AttnPlan&, const AttnArgs&, cudaStream_t) {
    return set_error(D2SD_ERR_UNSUPPORTED, "tcgen05 prefix pass not built");
}

}  // namespace d2sd
