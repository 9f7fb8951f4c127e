// C-ABI entry points, part 2: best_logp_grad, chain state, sampler dispatch, whitening, adaptation.
#include <cmath>
#include <cstring>

#include "best_internal.h"
#include "tc_fused.h"

using namespace best;

namespace {

struct DevBuf {  // RAII scratch
  void* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
  int alloc(size_t bytes) {
    if (cudaMalloc(&p, bytes ? bytes : 1) != cudaSuccess) {
      cudaGetLastError();
      set_error("cudaMalloc failed");
      return BEST_ERR_ALLOC;
    }
    return BEST_OK;
  }
};

// Gradient cache only (MH / AIES leave it stale): the cached log pi is NOT rewritten, so a read-back between
// two step calls cannot change the chain (1 x N steps == k x N/k steps bit for bit, with or without get()).
int refresh_grad(best_ctx* ctx, best_state* st, cudaStream_t s) {
  if (ctx->precision == BEST_PREC_BF16) {
    BEST_TRY(tc_eval_state(ctx, st, st->p_logp, st->grad, s));
  } else {
    BEST_TRY(eval_target_soa(ctx, st->theta, st->B, st->B, st->p_logp, st->grad, s));
    st->n_evals += (uint64_t)st->B;
  }
  st->grad_valid = true;
  return BEST_OK;
}

int refresh_cache(best_ctx* ctx, best_state* st, cudaStream_t s) {
  if (ctx->precision == BEST_PREC_BF16) return tc_state_init(ctx, st, s);
  BEST_TRY(eval_target_soa(ctx, st->theta, st->B, st->B, st->logp, st->grad, s));
  st->grad_valid = true;
  st->n_evals += (uint64_t)st->B;
  return BEST_OK;
}

int check_step_args(best_ctx* ctx, best_state* st, int64_t n, const float* trace, int thin) {
  if (!ctx || !st || st->ctx != ctx) { set_error("step: bad ctx/state"); return BEST_ERR_ARG; }
  if (n < 0) { set_error("step: n_steps < 0"); return BEST_ERR_ARG; }
  if (trace && thin > 0 && !is_device_ptr(trace)) { set_error("step: trace must be a device pointer"); return BEST_ERR_ARG; }
  return BEST_OK;
}

enum { M_MH = 0, M_MALA = 1, M_HMC = 2, M_AIES = 3 };

}  // namespace

namespace {
__global__ void k_sum_accept(const unsigned long long* __restrict__ n_accept, int64_t B,
                             unsigned long long* __restrict__ out) {
  unsigned long long s = 0;
  for (int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; c < B; c += (int64_t)gridDim.x * blockDim.x)
    s += n_accept[c];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0 && s) atomicAdd(out, s);
}

int total_accepts(best_state* st, unsigned long long* dev_tmp, unsigned long long* out, cudaStream_t s) {
  BEST_CUDA(cudaMemsetAsync(dev_tmp, 0, sizeof(unsigned long long), s));
  const int nb = (int)((st->B + 255) / 256 < 1024 ? (st->B + 255) / 256 : 1024);
  k_sum_accept<<<nb, 256, 0, s>>>(st->n_accept, st->B, dev_tmp);
  count_launch();
  BEST_CUDA(cudaMemcpyAsync(out, dev_tmp, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s));
  BEST_CUDA(cudaStreamSynchronize(s));
  return BEST_OK;
}
}  // namespace

extern "C" {

int best_logp_grad(best_ctx* ctx, const float* theta, int64_t n, float* logp, float* grad,
                   void* stream) {
  if (!ctx || n < 0) { set_error("best_logp_grad: bad argument"); return BEST_ERR_ARG; }
  if (n == 0) return BEST_OK;
  if (!theta || !logp) { set_error("best_logp_grad: NULL buffer"); return BEST_ERR_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  const int d = ctx->d;
  const bool th_dev = is_device_ptr(theta), lp_dev = is_device_ptr(logp);
  const bool g_dev = grad ? is_device_ptr(grad) : true;
  DevBuf b_th, b_lp, b_g;
  const float* th_d = theta;
  float* lp_d = logp;
  float* g_d = grad;
  if (!th_dev) {
    BEST_TRY(b_th.alloc(sizeof(float) * n * d));
    BEST_CUDA(cudaMemcpyAsync(b_th.p, theta, sizeof(float) * n * d, cudaMemcpyHostToDevice, s));
    th_d = (const float*)b_th.p;
  }
  if (!lp_dev) { BEST_TRY(b_lp.alloc(sizeof(float) * n)); lp_d = (float*)b_lp.p; }
  if (grad && !g_dev) { BEST_TRY(b_g.alloc(sizeof(float) * n * d)); g_d = (float*)b_g.p; }

  if (ctx->precision == BEST_PREC_BF16) {
    BEST_TRY(tc_logp_grad(ctx, th_d, n, lp_d, g_d, s));
  } else {
    // SoA fp64 staging [theta | grad | logp] in the context's grow-only scratch (no allocation per call)
    const size_t need = sizeof(double) * (size_t)n * (2 * (size_t)d + 1);
    if (need > ctx->lg_scratch_bytes) {
      BEST_CUDA(cudaStreamSynchronize(s));
      cudaFree(ctx->lg_scratch);
      ctx->lg_scratch = nullptr; ctx->lg_scratch_bytes = 0;
      if (cudaMalloc(&ctx->lg_scratch, need) != cudaSuccess) { cudaGetLastError(); set_error("cudaMalloc failed"); return BEST_ERR_ALLOC; }
      ctx->lg_scratch_bytes = need;
    }
    double* soa_th = (double*)ctx->lg_scratch;
    double* soa_g = soa_th + (size_t)n * d;
    double* lp64 = soa_g + (size_t)n * d;
    BEST_TRY(rows_f32_to_soa_f64(th_d, soa_th, n, d, n, s));
    BEST_TRY(eval_target_soa(ctx, soa_th, n, n, lp64, grad ? soa_g : nullptr, s));
    BEST_TRY(soa_f64_to_rows_f32(lp64, lp_d, n, 1, n, s));
    if (grad) BEST_TRY(soa_f64_to_rows_f32(soa_g, g_d, n, d, n, s));
  }
  if (!lp_dev) BEST_CUDA(cudaMemcpyAsync(logp, lp_d, sizeof(float) * n, cudaMemcpyDeviceToHost, s));
  if (grad && !g_dev) BEST_CUDA(cudaMemcpyAsync(grad, g_d, sizeof(float) * n * d, cudaMemcpyDeviceToHost, s));
  if (!th_dev || !lp_dev || (grad && !g_dev)) BEST_CUDA(cudaStreamSynchronize(s));
  return BEST_OK;
}

int best_state_create(best_ctx* ctx, int64_t n_chains, const float* theta0, void* stream,
                      best_state** out) {
  if (!ctx || !theta0 || !out || n_chains < 1 || n_chains > (int64_t)1 << 31) {
    set_error("best_state_create: bad argument");
    return BEST_ERR_ARG;
  }
  *out = nullptr;
  best_state* st = new best_state();
  st->ctx = ctx;
  st->B = n_chains;
  const size_t B = (size_t)n_chains, d = (size_t)ctx->d;
  int rc = BEST_OK;
  auto A = [&](double** p, size_t n) { if (!rc) rc = dev_alloc(p, n); };
  A(&st->theta, B * d); A(&st->grad, B * d); A(&st->logp, B);
  A(&st->p_theta, B * d); A(&st->p_grad, B * d); A(&st->p_logp, B);
  A(&st->q, B * d); A(&st->h0, B); A(&st->last_la, B);
  if (!rc) rc = dev_alloc(&st->n_accept, B);
  if (!rc) rc = dev_alloc(&st->stage, B * d);
  if (rc) { best_state_destroy(st); return rc; }
  cudaMemset(st->n_accept, 0, sizeof(unsigned long long) * B);
  cudaMemset(st->last_la, 0, sizeof(double) * B);
  rc = best_state_set(st, theta0, 0, stream);
  if (rc) { best_state_destroy(st); return rc; }
  *out = st;
  return BEST_OK;
}

void best_state_destroy(best_state* st) {
  if (!st) return;
  cudaFree(st->theta); cudaFree(st->grad); cudaFree(st->logp);
  cudaFree(st->p_theta); cudaFree(st->p_grad); cudaFree(st->p_logp);
  cudaFree(st->q); cudaFree(st->h0); cudaFree(st->last_la); cudaFree(st->n_accept); cudaFree(st->stage);
  adapt_free(st);
  delete st;
}

int best_state_set(best_state* st, const float* theta, uint64_t step, void* stream) {
  if (!st || !theta) { set_error("best_state_set: bad argument"); return BEST_ERR_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  best_ctx* ctx = st->ctx;
  const size_t nb = sizeof(float) * st->B * ctx->d;
  const float* src = theta;
  if (!is_device_ptr(theta)) {
    BEST_CUDA(cudaMemcpyAsync(st->stage, theta, nb, cudaMemcpyHostToDevice, s));
    src = st->stage;
  }
  BEST_TRY(rows_f32_to_soa_f64(src, st->theta, st->B, ctx->d, st->B, s));
  st->step = step;
  BEST_TRY(refresh_cache(ctx, st, s));
  BEST_CUDA(cudaStreamSynchronize(s));
  return BEST_OK;
}

int best_state_get(best_state* st, float* theta, float* logp, float* grad, uint64_t* step,
                   uint64_t* n_accept, uint64_t* n_evals, void* stream) {
  if (!st) { set_error("best_state_get: NULL state"); return BEST_ERR_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  best_ctx* ctx = st->ctx;
  const int64_t B = st->B;
  const int d = ctx->d;
  if (grad && !st->grad_valid) BEST_TRY(refresh_grad(ctx, st, s));
  if (theta) {
    BEST_TRY(soa_f64_to_rows_f32(st->theta, st->stage, B, d, B, s));
    BEST_CUDA(cudaMemcpyAsync(theta, st->stage, sizeof(float) * B * d, cudaMemcpyDeviceToHost, s));
    BEST_CUDA(cudaStreamSynchronize(s));
  }
  if (grad) {
    BEST_TRY(soa_f64_to_rows_f32(st->grad, st->stage, B, d, B, s));
    BEST_CUDA(cudaMemcpyAsync(grad, st->stage, sizeof(float) * B * d, cudaMemcpyDeviceToHost, s));
    BEST_CUDA(cudaStreamSynchronize(s));
  }
  if (logp) {
    BEST_TRY(soa_f64_to_rows_f32(st->logp, st->stage, B, 1, B, s));
    BEST_CUDA(cudaMemcpyAsync(logp, st->stage, sizeof(float) * B, cudaMemcpyDeviceToHost, s));
  }
  if (n_accept)
    BEST_CUDA(cudaMemcpyAsync(n_accept, st->n_accept, sizeof(uint64_t) * B, cudaMemcpyDeviceToHost, s));
  BEST_CUDA(cudaStreamSynchronize(s));
  if (step) *step = st->step;
  if (n_evals) *n_evals = st->n_evals;
  return BEST_OK;
}

int best_state_get_f64(best_state* st, double* theta, double* logp, double* grad, void* stream) {
  if (!st) { set_error("best_state_get_f64: NULL state"); return BEST_ERR_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  const int64_t B = st->B;
  const int d = st->ctx->d;
  BEST_CUDA(cudaStreamSynchronize(s));
  std::vector<double> tmp((size_t)B * d);
  auto fetch = [&](const double* src, double* dst) -> int {
    BEST_CUDA(cudaMemcpy(tmp.data(), src, sizeof(double) * B * d, cudaMemcpyDeviceToHost));
    for (int64_t c = 0; c < B; ++c)
      for (int i = 0; i < d; ++i) dst[c * d + i] = tmp[(size_t)i * B + c];
    return BEST_OK;
  };
  if (theta) BEST_TRY(fetch(st->theta, theta));
  if (grad) {
    if (!st->grad_valid) {
      BEST_TRY(refresh_grad(st->ctx, st, s));
      BEST_CUDA(cudaStreamSynchronize(s));
    }
    BEST_TRY(fetch(st->grad, grad));
  }
  if (logp) BEST_CUDA(cudaMemcpy(logp, st->logp, sizeof(double) * B, cudaMemcpyDeviceToHost));
  return BEST_OK;
}

int best_state_last_log_alpha(best_state* st, double* log_alpha, void* stream) {
  if (!st || !log_alpha) { set_error("best_state_last_log_alpha: bad argument"); return BEST_ERR_ARG; }
  BEST_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  BEST_CUDA(cudaMemcpy(log_alpha, st->last_la, sizeof(double) * st->B, cudaMemcpyDeviceToHost));
  return BEST_OK;
}

static int run_step(best_ctx* ctx, best_state* st, int method, int64_t n, uint64_t seed, float eps,
                    int nl, float* trace, int thin, void* stream, bool de = false) {
  BEST_TRY(check_step_args(ctx, st, n, trace, thin));
  cudaStream_t s = (cudaStream_t)stream;
  if (method != M_AIES && !(eps > 0.f)) { set_error("step: eps must be > 0"); return BEST_ERR_ARG; }
  if (method == M_HMC && nl < 1) { set_error("hmc: n_leapfrog must be >= 1"); return BEST_ERR_ARG; }
  if (method == M_AIES && de) {
    if (!(eps >= 0.f)) { set_error("aies_de: sigma_gamma must be >= 0"); return BEST_ERR_ARG; }
    if (st->B < 4 || (st->B & 1)) { set_error("aies_de: walker count must be even and >= 4"); return BEST_ERR_ARG; }
  } else if (method == M_AIES) {
    if (!(eps > 1.f)) { set_error("aies: a must be > 1"); return BEST_ERR_ARG; }
    if (st->B < 2 || (st->B & 1)) { set_error("aies: walker count must be even and >= 2"); return BEST_ERR_ARG; }
  }
  if (method == M_AIES && st->aies_fn && trace) {
    set_error("ensemble move sharded over ranks (best_set_aies_exchange): no trace, read the state instead");
    return BEST_ERR_ARG;
  }
  if (n == 0) return BEST_OK;
  int rc;
  if (ctx->precision == BEST_PREC_BF16) {
    rc = tc_step(ctx, st, method, n, seed, eps, nl, trace, thin, s, de);
  } else {
    if ((method == M_MALA || method == M_HMC) && !st->grad_valid) {
      BEST_TRY(eval_target_soa(ctx, st->theta, st->B, st->B, st->logp, st->grad, s));
      st->grad_valid = true;
    }
    switch (method) {
      case M_MH: rc = step_mh(ctx, st, n, seed, eps, trace, thin, s); st->grad_valid = false; break;
      case M_MALA: rc = step_mala(ctx, st, n, seed, eps, trace, thin, s); break;
      case M_HMC: rc = step_hmc(ctx, st, n, seed, eps, nl, trace, thin, s); break;
      default: rc = step_aies(ctx, st, n, seed, eps, trace, thin, s, de); st->grad_valid = false; break;
    }
  }
  if (rc) return rc;
  st->step += (uint64_t)n;
  st->n_evals += (uint64_t)st->B * (uint64_t)n * (uint64_t)(method == M_HMC ? nl : 1);
  return BEST_OK;
}

int best_step_mh(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float eps,
                 float* trace_dev, int32_t thin, void* stream) {
  return run_step(ctx, st, M_MH, n_steps, seed, eps, 0, trace_dev, thin, stream);
}
int best_step_mala(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float eps,
                   float* trace_dev, int32_t thin, void* stream) {
  return run_step(ctx, st, M_MALA, n_steps, seed, eps, 0, trace_dev, thin, stream);
}
int best_step_hmc(best_ctx* ctx, best_state* st, int64_t n_traj, uint64_t seed, float eps,
                  int32_t n_leapfrog, float* trace_dev, int32_t thin, void* stream) {
  return run_step(ctx, st, M_HMC, n_traj, seed, eps, n_leapfrog, trace_dev, thin, stream);
}
int best_step_aies(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float a,
                   float* trace_dev, int32_t thin, void* stream) {
  return run_step(ctx, st, M_AIES, n_steps, seed, a, 0, trace_dev, thin, stream);
}
int best_step_aies_de(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float sigma_gamma,
                      float* trace_dev, int32_t thin, void* stream) {
  return run_step(ctx, st, M_AIES, n_steps, seed, sigma_gamma, 0, trace_dev, thin, stream, true);
}

int best_set_adaptation(best_ctx* ctx, best_state* st, int32_t adapt_every, double jitter) {
  if (!ctx || !st || st->ctx != ctx || adapt_every < 0 || !(jitter >= 0.0)) {
    set_error("best_set_adaptation: bad argument");
    return BEST_ERR_ARG;
  }
  BEST_CUDA(cudaDeviceSynchronize());   // work in flight on any stream is ordered before the window opens
  st->adapt_every = adapt_every;
  st->jitter = jitter;
  if (adapt_every > 0) {
    BEST_TRY(adapt_reset(ctx, st, 0));
    BEST_CUDA(cudaDeviceSynchronize());
  }
  return BEST_OK;
}

int best_set_adaptation_exchange(best_state* st, best_exchange_fn fn, void* user, int32_t world_size) {
  if (!st || world_size < 1 || world_size > 4096) {
    set_error("best_set_adaptation_exchange: bad argument");
    return BEST_ERR_ARG;
  }
  BEST_CUDA(cudaDeviceSynchronize());
  st->xchg_fn = nullptr;
  cudaFree(st->xchg_buf);
  st->xchg_buf = nullptr;
  if (fn) {
    const int d = st->ctx->d;
    const size_t np = 1 + 2 * (size_t)d + (size_t)d * d;
    BEST_TRY(dev_alloc(&st->xchg_buf, np * (size_t)(1 + world_size)));
    st->xchg_fn = fn; st->xchg_user = user; st->xchg_world = world_size;
  }
  return BEST_OK;
}

int best_set_aies_exchange(best_state* st, best_exchange_fn fn, void* user, int32_t rank, int32_t world_size) {
  if (!st || world_size < 1 || rank < 0 || rank >= world_size || (st->B & 1) ||
      (fn && ((st->B / 2) % world_size != 0 || st->B / 2 / world_size < 1))) {
    set_error("best_set_aies_exchange: bad argument (the half-ensemble must divide evenly over the ranks)");
    return BEST_ERR_ARG;
  }
  BEST_CUDA(cudaDeviceSynchronize());
  st->aies_fn = nullptr;
  cudaFree(st->aies_buf);
  st->aies_buf = nullptr;
  if (fn) {
    const size_t n = (size_t)(st->ctx->d + 1) * (size_t)(st->B / 2 / world_size);
    BEST_TRY(dev_alloc(&st->aies_buf, n * (size_t)(1 + world_size)));
    st->aies_fn = fn; st->aies_user = user; st->aies_rank = rank; st->aies_world = world_size;
  }
  return BEST_OK;
}

int best_state_set_chain_offset(best_state* st, uint64_t chain0) {
  if (!st || chain0 + (uint64_t)st->B > ((uint64_t)1 << 32)) {
    set_error("best_state_set_chain_offset: chain0 + n_chains must not exceed 2^32");
    return BEST_ERR_ARG;
  }
  st->chain0 = chain0;
  return BEST_OK;
}

int best_adapt_stats(best_ctx* ctx, int64_t* n_updates, int64_t* n_failures) {
  if (!ctx) { set_error("best_adapt_stats: NULL ctx"); return BEST_ERR_ARG; }
  int64_t h[2];
  BEST_CUDA(cudaDeviceSynchronize());
  BEST_CUDA(cudaMemcpy(h, ctx->adapt_counts, sizeof(h), cudaMemcpyDeviceToHost));
  if (n_updates) *n_updates = h[0];
  if (n_failures) *n_failures = h[1];
  return BEST_OK;
}

int best_get_whitening(best_ctx* ctx, double* L_host) {
  if (!ctx || !L_host) { set_error("best_get_whitening: bad argument"); return BEST_ERR_ARG; }
  BEST_CUDA(cudaDeviceSynchronize());
  BEST_CUDA(cudaMemcpy(L_host, ctx->Lraw_dev, sizeof(double) * ctx->d * ctx->d, cudaMemcpyDeviceToHost));
  return BEST_OK;
}

// L_dev = L_raw diag(s): the factor every step kernel applies (columns scaled, still lower triangular)
static int refresh_scaled_whitening(best_ctx* ctx) {
  const int d = ctx->d;
  std::vector<double> L((size_t)d * d), s((size_t)d);
  BEST_CUDA(cudaMemcpy(L.data(), ctx->Lraw_dev, sizeof(double) * d * d, cudaMemcpyDeviceToHost));
  BEST_CUDA(cudaMemcpy(s.data(), ctx->scale_dev, sizeof(double) * d, cudaMemcpyDeviceToHost));
  for (int i = 0; i < d; ++i)
    for (int j = 0; j < d; ++j) L[(size_t)i * d + j] *= s[j];
  BEST_CUDA(cudaMemcpy(ctx->L_dev, L.data(), sizeof(double) * d * d, cudaMemcpyHostToDevice));
  return BEST_OK;
}

int best_set_step_scale(best_ctx* ctx, const double* s_host) {
  if (!ctx) { set_error("best_set_step_scale: NULL ctx"); return BEST_ERR_ARG; }
  const int d = ctx->d;
  std::vector<double> s((size_t)d, 1.0);
  if (s_host)
    for (int i = 0; i < d; ++i) {
      if (!(s_host[i] > 0.0) || !std::isfinite(s_host[i])) {
        set_error("best_set_step_scale: factors must be positive and finite");
        return BEST_ERR_ARG;
      }
      s[i] = s_host[i];
    }
  BEST_CUDA(cudaDeviceSynchronize());
  BEST_CUDA(cudaMemcpy(ctx->scale_dev, s.data(), sizeof(double) * d, cudaMemcpyHostToDevice));
  return refresh_scaled_whitening(ctx);
}

int best_set_hard_box(best_ctx* ctx, int32_t on) {
  if (!ctx) { set_error("best_set_hard_box: NULL ctx"); return BEST_ERR_ARG; }
  if (on && !ctx->tgt.has_box) { set_error("best_set_hard_box: the target has no box"); return BEST_ERR_ARG; }
  BEST_CUDA(cudaDeviceSynchronize());
  ctx->tgt.hard_box = on ? 1 : 0;
  return BEST_OK;
}

int best_set_whitening(best_ctx* ctx, const double* L_host) {
  if (!ctx || !L_host) { set_error("best_set_whitening: bad argument"); return BEST_ERR_ARG; }
  const int d = ctx->d;
  std::vector<double> L((size_t)d * d, 0.0);
  for (int i = 0; i < d; ++i)
    for (int j = 0; j <= i; ++j) {
      L[(size_t)i * d + j] = L_host[(size_t)i * d + j];
      if (i == j && !(L_host[(size_t)i * d + j] > 0.0)) {
        set_error("best_set_whitening: diag(L) must be positive");
        return BEST_ERR_NOT_SPD;
      }
    }
  BEST_CUDA(cudaDeviceSynchronize());
  BEST_CUDA(cudaMemcpy(ctx->Lraw_dev, L.data(), sizeof(double) * d * d, cudaMemcpyHostToDevice));
  return refresh_scaled_whitening(ctx);
}

int best_burn_in(best_ctx* ctx, best_state* st, int32_t method, int32_t n_iter, int64_t n_steps,
                 int64_t n_adapt, int64_t block, uint64_t seed, float* eps_inout, float target_accept,
                 int32_t n_leapfrog, double jitter, float* best_theta, double* best_logp,
                 float* eps_hist, void* stream) {
  if (!ctx || !st || st->ctx != ctx || !eps_inout) { set_error("best_burn_in: bad ctx/state/eps"); return BEST_ERR_ARG; }
  if (method != BEST_METHOD_MH && method != BEST_METHOD_MALA && method != BEST_METHOD_HMC) {
    set_error("best_burn_in: method must be MH, MALA or HMC (no burn-in loop for AIES)");
    return BEST_ERR_ARG;
  }
  if (n_iter < 0 || n_steps < 0 || n_adapt < 0 || n_adapt > n_steps || (n_adapt > 0 && block < 1) ||
      !(target_accept > 0.f && target_accept < 1.f) || !(*eps_inout > 0.f) || !(jitter >= 0.0)) {
    set_error("best_burn_in: bad schedule / target_accept / eps / jitter");
    return BEST_ERR_ARG;
  }
  cudaStream_t s = (cudaStream_t)stream;
  const int m_int = method == BEST_METHOD_MH ? M_MH : method == BEST_METHOD_MALA ? M_MALA : M_HMC;
  constexpr double kGamma = 0.05, kT0 = 10.0, kKappa = 0.75;
  DevBuf tmp;
  BEST_TRY(tmp.alloc(sizeof(unsigned long long)));
  unsigned long long* dtmp = (unsigned long long*)tmp.p;
  float eps = *eps_inout;
  double best_lp = -INFINITY;
  std::vector<double> lp_host((size_t)st->B);
  int64_t nh = 0;
  st->adapt_every = 0;
  for (int it = 0; it < n_iter; ++it) {
    if (n_adapt > 0) {  // (1) dual averaging on the ensemble acceptance fraction
      const double mu = std::log(10.0 * (double)eps);
      double hbar = 0.0, logeps_bar = 0.0, cur = (double)eps;
      int64_t done = 0;
      int m = 0;
      while (done < n_adapt) {
        const int64_t nb = (block < n_adapt - done) ? block : (n_adapt - done);
        unsigned long long a0 = 0, a1 = 0;
        BEST_TRY(total_accepts(st, dtmp, &a0, s));
        const float cur32 = (float)cur;
        if (eps_hist) eps_hist[nh] = cur32;
        ++nh;
        BEST_TRY(run_step(ctx, st, m_int, nb, seed, cur32, n_leapfrog, nullptr, 0, stream));
        BEST_TRY(total_accepts(st, dtmp, &a1, s));
        const double alpha = (double)(a1 - a0) / ((double)st->B * (double)nb);
        ++m;
        hbar = (1.0 - 1.0 / (m + kT0)) * hbar + ((double)target_accept - alpha) / (m + kT0);
        const double logeps = mu - std::sqrt((double)m) / kGamma * hbar;
        const double eta = std::pow((double)m, -kKappa);
        logeps_bar = eta * logeps + (1.0 - eta) * logeps_bar;
        cur = std::exp(logeps);
        done += nb;
      }
      eps = (float)std::exp(logeps_bar);
    }
    const int64_t win = n_steps - n_adapt;
    if (win > 0) {  // (2) one covariance window -> whitening update on the device
      if (win > INT32_MAX) { set_error("best_burn_in: window too long"); return BEST_ERR_ARG; }
      BEST_TRY(best_set_adaptation(ctx, st, (int32_t)win, jitter));
      const int rc = run_step(ctx, st, m_int, win, seed, eps, n_leapfrog, nullptr, 0, stream);
      st->adapt_every = 0;
      if (rc) return rc;
    }
    // (3) best fit over the ensemble (first chain with the largest cached log pi)
    BEST_CUDA(cudaStreamSynchronize(s));
    BEST_CUDA(cudaMemcpy(lp_host.data(), st->logp, sizeof(double) * st->B, cudaMemcpyDeviceToHost));
    int64_t arg = 0;
    for (int64_t c = 1; c < st->B; ++c)
      if (lp_host[c] > lp_host[arg]) arg = c;
    if (st->B > 0 && lp_host[arg] > best_lp) {
      best_lp = lp_host[arg];
      if (best_theta)
        for (int i = 0; i < ctx->d; ++i) {
          double v;
          BEST_CUDA(cudaMemcpy(&v, st->theta + (size_t)i * st->B + arg, sizeof(double), cudaMemcpyDeviceToHost));
          best_theta[i] = (float)v;
        }
    }
  }
  *eps_inout = eps;
  if (best_logp) *best_logp = best_lp;
  return BEST_OK;
}

}  // extern "C"
