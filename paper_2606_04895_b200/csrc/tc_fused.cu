// bf16 tensor-core path — placeholder until the tcgen05 kernel lands (next commit).
#include "tc_fused.h"

namespace best {
int tc_plan_create(best_ctx*, const best_config*) {
  set_error("BEST_PREC_BF16: tensor-core path not built yet");
  return BEST_ERR_UNSUPPORTED;
}
void tc_plan_destroy(best_ctx*) {}
int tc_logp_grad(best_ctx*, const float*, int64_t, float*, float*, cudaStream_t) { return BEST_ERR_UNSUPPORTED; }
int tc_state_init(best_ctx*, best_state*, cudaStream_t) { return BEST_ERR_UNSUPPORTED; }
int tc_step(best_ctx*, best_state*, int, int64_t, uint64_t, float, int, float*, int, cudaStream_t) {
  return BEST_ERR_UNSUPPORTED;
}
}  // namespace best
