// Internal declarations of libbest.so (host side).  Not part of the public boundary.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/best.h"

namespace best {

void set_error(const std::string& msg);
extern std::atomic<uint64_t> g_launches;
inline void count_launch(uint64_t n = 1) { g_launches.fetch_add(n, std::memory_order_relaxed); }

#define BEST_CUDA(expr)                                                                    \
  do {                                                                                     \
    cudaError_t _e = (expr);                                                               \
    if (_e != cudaSuccess) {                                                               \
      best::set_error(std::string(#expr) + ": " + cudaGetErrorString(_e));                 \
      return BEST_ERR_CUDA;                                                                \
    }                                                                                      \
  } while (0)

#define BEST_TRY(expr)           \
  do {                           \
    int _rc = (expr);            \
    if (_rc != BEST_OK) return _rc; \
  } while (0)

inline bool is_device_ptr(const void* p) {
  if (!p) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

template <typename T>
int dev_alloc(T** p, size_t n) {
  *p = nullptr;
  if (n == 0) n = 1;
  if (cudaMalloc((void**)p, sizeof(T) * n) != cudaSuccess) {
    cudaGetLastError();
    set_error("cudaMalloc failed");
    return BEST_ERR_ALLOC;
  }
  return BEST_OK;
}

constexpr int kMaxD = 32;
constexpr int64_t kEvalChunk = 16384;  // chains per emulator pass on the fp32 path (bounds scratch)

// Target terms that every kernel needs by value (device pointers inside).
struct TargetDev {
  int d;
  int has_gauss, has_box;
  const double* mu;   // [d]
  const double* R;    // [d*d] upper triangular, Sigma_inv = R^T R
  const double* lo;   // [d]
  const double* hi;   // [d]
  double pen_kappa, pen_gamma;
  int banana_i, banana_j;
  double banana_sigma;
  double mlp_scale;
  int has_mlp;
  int hard_box;  // 8(f)#1: log pi = -inf outside [lo, hi] instead of the smooth penalty
};

struct TcPlan;  // bf16 tensor-core path (tc_fused.cu)
}  // namespace best
namespace best {
struct Tc32Plan;  // fp32-accurate split-operand tensor-core GEMMs of the exact path (emulator_tc32.cu)

}  // namespace best

struct best_ctx {
  int d = 0, dp = 0;  // dp = d rounded up to 4 (row pitch of MLP input / theta-gradient)
  int n_affine = 0;
  std::vector<int> widths, wp;  // wp: widths padded to multiples of 4 (wp[0] = dp, last = 1)
  int activation = 0;
  int precision = 0;
  best::TargetDev tgt{};
  // fp32 emulator weights, zero padded: W[k] [wp[k+1]][wp[k]], b[k] [wp[k+1]]
  std::vector<float*> W, b;
  double* dev_consts = nullptr;  // mu | R | lo | hi | L  (5 blocks)
  double* L_dev = nullptr;       // [d*d] lower triangular, updated on device by adaptation: L_raw * diag(step scale)
  double* Lraw_dev = nullptr;    // [d*d] the whitening factor itself | [d] per-dimension step factors (8(f)#1)
  double* scale_dev = nullptr;   // = Lraw_dev + d*d
  // fp32 emulator scratch (sized for scratch_n chains)
  int64_t scratch_n = 0;
  float* X0 = nullptr;            // [n][dp]
  std::vector<float*> H, Dact;    // per hidden layer [n][wp[k+1]]
  float* delta[2] = {nullptr, nullptr};
  float* mlp_out = nullptr;       // [n]
  float* mlp_grad = nullptr;      // [n][dp]
  int64_t* adapt_counts = nullptr;  // device [2]: whitening updates, failures (A9)
  // best_logp_grad scratch on the exact path (grow-only; a context is driven from one stream at a time)
  void* lg_scratch = nullptr;
  size_t lg_scratch_bytes = 0;
  best::TcPlan* tc = nullptr;
  best::Tc32Plan* tc32 = nullptr;
};

struct best_state {
  best_ctx* ctx = nullptr;
  int64_t B = 0;
  uint64_t step = 0;
  uint64_t n_evals = 0;
  bool grad_valid = true;  // AIES does not maintain the cached gradient
  // SoA [d][B] fp64
  double *theta = nullptr, *grad = nullptr, *logp = nullptr;
  double *p_theta = nullptr, *p_grad = nullptr, *p_logp = nullptr;
  double *q = nullptr, *h0 = nullptr;
  double* last_la = nullptr;
  unsigned long long* n_accept = nullptr;
  float* stage = nullptr;  // [B*d] fp32 row-major staging for best_state_set / _get (no allocation per call)
  uint64_t chain0 = 0;     // Philox chain id of chain 0 (best_state_set_chain_offset)
  // covariance adaptation (A9) -- per STATE: the window of one state never sees another state's samples
  int adapt_every = 0;
  double jitter = 1e-6;
  int64_t win_steps = 0;          // steps accumulated in the current window
  double* cov_acc = nullptr;      // [cov_blocks][1 + d + d*d] per-block partial sums (fp64): count | sums | products
  int cov_blocks = 0;
  double* cov_ref = nullptr;      // [d] shift (chain 0's position when the window opened)
  // tensor path: two fp32 row buffers [win_cap_steps][B][d] that the persistent kernel writes in turn; the Gram
  // kernel of a segment runs on `side`, concurrently with the next segment's persistent launch
  float* win_buf[2] = {nullptr, nullptr};
  int64_t win_cap_steps = 0;      // steps per segment of the current window
  int64_t win_cap_alloc = 0;      // steps the buffers were allocated for
  int win_flip = 0;
  cudaStream_t side = nullptr;
  cudaEvent_t ev_seg[2] = {nullptr, nullptr}, ev_gram[2] = {nullptr, nullptr};
  // multi-GPU: the window's sums of ALL ranks feed the covariance (best_set_adaptation_exchange)
  best_exchange_fn xchg_fn = nullptr;
  void* xchg_user = nullptr;
  int xchg_world = 1;
  double* xchg_buf = nullptr;     // [1 + world] packets of 1 + 2d + d*d doubles: own packet, then the gathered ones
  // sharded ensemble moves (best_set_aies_exchange): every rank holds the whole ensemble, updates walkers
  // [rank * cnt, +cnt) of each half (cnt = B / 2 / world) and all-gathers them after every half-step
  best_exchange_fn aies_fn = nullptr;
  void* aies_user = nullptr;
  int aies_rank = 0, aies_world = 1;
  double* aies_buf = nullptr;     // [(1 + world)][d + 1][cnt]: own slice (theta rows, then log pi), then the gathered ones
};

namespace best {

// fp32 emulator (emulator_fp32.cu): MLP forward (+ input gradient) for n points.
// X0 = ctx->X0 must already hold the inputs [n][dp]; results in ctx->mlp_out / ctx->mlp_grad.
int mlp_fp32_reserve(best_ctx* ctx, int64_t n);
int mlp_fp32_run(best_ctx* ctx, int64_t n, bool want_grad, cudaStream_t s);
// emulator_tc32.cu: the same GEMMs on the tensor cores with fp16-pair split operands (fp32-accurate)
int tc32_plan_create(best_ctx* ctx, const best_config* cfg);
void tc32_plan_destroy(best_ctx* ctx);
int tc32_gemm(best_ctx* ctx, bool forward, int layer, const float* A, int lda, float* C, int ldc, int M,
              const float* bias, float* aux, int ldaux, int epi, cudaStream_t s);

// Full target for SoA fp64 inputs (samplers.cu): theta [d][ld] (first n columns used).
int eval_target_soa(best_ctx* ctx, const double* theta, int64_t ld, int64_t n, double* logp,
                    double* grad /*nullable, [d][ld]*/, cudaStream_t s);

int step_mh(best_ctx*, best_state*, int64_t, uint64_t, double, float*, int, cudaStream_t);
int step_mala(best_ctx*, best_state*, int64_t, uint64_t, double, float*, int, cudaStream_t);
int step_hmc(best_ctx*, best_state*, int64_t, uint64_t, double, int, float*, int, cudaStream_t);
int step_aies(best_ctx*, best_state*, int64_t, uint64_t, double, float*, int, cudaStream_t, bool de = false);
int adapt_reset(best_ctx* ctx, best_state* st, cudaStream_t s);
// sharded ensemble moves: all-gather the walkers [half0 + rank * cnt, +cnt) that this rank has just updated
int aies_exchange(best_ctx* ctx, best_state* st, int64_t half0, cudaStream_t s);
void adapt_free(best_state* st);
// exact path, after step index t of a call: trace slot (every `thin` steps) and covariance accumulation / update
int after_step(best_ctx* ctx, best_state* st, int64_t t, float* trace, int thin, bool adapt, cudaStream_t s);
// tensor path: fold `n_steps` slots of fp32 rows [n_steps][B][d] (every post-accept state of a segment) into
// the window sums; closes the window (covariance -> Cholesky -> whitening swap, on device) when it is complete
int adapt_window_rows(best_ctx* ctx, best_state* st, int buf, int64_t n_steps, cudaStream_t s);
// the window buffer the next segment may write (waits, on `s`, until its previous contents have been folded)
int adapt_acquire_buffer(best_state* st, cudaStream_t s, int* buf);

// layout helpers (samplers.cu)
int rows_f32_to_soa_f64(const float* rows_dev, double* soa, int64_t n, int d, int64_t ld, cudaStream_t s);
int soa_f64_to_rows_f32(const double* soa, float* rows_dev, int64_t n, int d, int64_t ld, cudaStream_t s);

}  // namespace best
