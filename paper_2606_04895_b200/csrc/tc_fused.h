// bf16 tensor-core path (tcgen05 / TMEM / bulk-copy weight streaming), see tc_fused.cu.
#pragma once
#include "best_internal.h"

namespace best {
int tc_plan_create(best_ctx* ctx, const best_config* cfg);
void tc_plan_destroy(best_ctx* ctx);
// log pi (+ gradient) for n points given as fp32 rows [n][d] on the device
int tc_logp_grad(best_ctx* ctx, const float* theta_rows, int64_t n, float* logp, float* grad,
                 cudaStream_t s);
int tc_state_init(best_ctx* ctx, best_state* st, cudaStream_t s);
// log pi / gradient at the state's theta into caller-chosen SoA fp64 buffers (does not touch the caches)
int tc_eval_state(best_ctx* ctx, best_state* st, double* logp_out, double* grad_out, cudaStream_t s);
int tc_step(best_ctx* ctx, best_state* st, int method, int64_t n_steps, uint64_t seed, float eps,
            int n_leapfrog, float* trace, int thin, cudaStream_t s, bool de = false);
}  // namespace best
