// Exact path (BEST_PREC_FP32): per-chain target terms (A1a, A1d, A1e), whitening (A2), Philox
// (A3), MH / MALA / HMC / AIES step kernels (A4-A8) and covariance adaptation (A9).
// One thread per chain; chain state is SoA [d][B] in fp64 so every access is coalesced.
#include "best_internal.h"
#include "device_math.cuh"

namespace best {
namespace {

constexpr int TPB = 128;
inline int nblocks(int64_t n, int tpb = TPB) { return (int)((n + tpb - 1) / tpb); }

// ---------------------------------------------------------------------------------------------
// layout helpers
// ---------------------------------------------------------------------------------------------
__global__ void k_rows_to_soa(const float* __restrict__ rows, double* __restrict__ soa, int64_t n,
                              int d, int64_t ld) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= n) return;
  for (int i = 0; i < d; ++i) soa[i * ld + c] = (double)rows[c * d + i];
}
__global__ void k_soa_to_rows(const double* __restrict__ soa, float* __restrict__ rows, int64_t n,
                              int d, int64_t ld) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= n) return;
  for (int i = 0; i < d; ++i) rows[c * d + i] = (float)soa[i * ld + c];
}

// MLP input rows (fp32, pitch dp, zero padded) from the SoA fp64 state
__global__ void k_prep_input(const double* __restrict__ theta, int64_t ld, int64_t n, int d, int dp,
                             float* __restrict__ X0) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= n) return;
  for (int i = 0; i < dp; ++i) X0[c * dp + i] = (i < d) ? (float)theta[i * ld + c] : 0.0f;
}

__device__ __forceinline__ double pen_f(double t, double& df) {
  if (t <= 40.0) { df = expm1(t); return df - t; }
  const double s40 = expm1(40.0);
  df = s40;
  return (s40 - 40.0) + s40 * (t - 40.0);
}

// log pi and gradient from the emulator outputs + Gaussian (via R), banana and box terms, fp64
__global__ void k_finish_target(TargetDev T, const double* __restrict__ theta, int64_t ld, int64_t n,
                                const float* __restrict__ mlp_out, const float* __restrict__ mlp_grad,
                                int dp, double* __restrict__ logp, double* __restrict__ grad) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= n) return;
  const int d = T.d;
  double th[kMaxD], g[kMaxD];
  for (int i = 0; i < d; ++i) { th[i] = theta[i * ld + c]; g[i] = 0.0; }
  double lp = 0.0;
  if (T.has_mlp) {
    lp += T.mlp_scale * (double)mlp_out[c];
    if (grad) for (int i = 0; i < d; ++i) g[i] += T.mlp_scale * (double)mlp_grad[c * dp + i];
  }
  if (T.has_gauss) {  // y = R (theta - mu); logp = -1/2 |y|^2; grad = -R^T y
    double r[kMaxD], y[kMaxD];
    for (int i = 0; i < d; ++i) r[i] = th[i] - T.mu[i];
    double q = 0.0;
    for (int i = 0; i < d; ++i) {
      double s = 0.0;
      for (int j = i; j < d; ++j) s += T.R[i * d + j] * r[j];
      y[i] = s;
      q += s * s;
    }
    lp += -0.5 * q;
    if (grad)
      for (int j = 0; j < d; ++j) {
        double s = 0.0;
        for (int i = 0; i <= j; ++i) s += T.R[i * d + j] * y[i];
        g[j] -= s;
      }
  }
  if (T.banana_i >= 0) {
    const double ti = th[T.banana_i], tj = th[T.banana_j];
    const double t = tj - ti * ti, s2 = T.banana_sigma * T.banana_sigma;
    lp += -t * t / (2.0 * s2);
    g[T.banana_j] += -t / s2;
    g[T.banana_i] += 2.0 * ti * t / s2;
  }
  if (T.has_box && T.hard_box) {  // 8(f)#1: -inf outside the box, no penalty term
    for (int i = 0; i < d; ++i)
      if (th[i] < T.lo[i] || th[i] > T.hi[i]) lp = -INFINITY;
  } else if (T.has_box) {
    double pen = 0.0;
    for (int i = 0; i < d; ++i) {
      const double lo = T.lo[i], hi = T.hi[i], width = hi - lo;
      double ex = 0.0, sgn = 0.0;
      if (th[i] < lo) { ex = lo - th[i]; sgn = -1.0; }
      else if (th[i] > hi) { ex = th[i] - hi; sgn = 1.0; }
      if (ex > 0.0) {
        double df;
        pen += pen_f(T.pen_gamma * ex / width, df);
        g[i] -= T.pen_kappa * df * T.pen_gamma / width * sgn;
      }
    }
    lp -= T.pen_kappa * pen;
  }
  logp[c] = lp;
  if (grad) for (int i = 0; i < d; ++i) grad[i * ld + c] = g[i];
}

}  // namespace

int rows_f32_to_soa_f64(const float* rows, double* soa, int64_t n, int d, int64_t ld, cudaStream_t s) {
  if (n == 0) return BEST_OK;
  k_rows_to_soa<<<nblocks(n), TPB, 0, s>>>(rows, soa, n, d, ld);
  count_launch();
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}
int soa_f64_to_rows_f32(const double* soa, float* rows, int64_t n, int d, int64_t ld, cudaStream_t s) {
  if (n == 0) return BEST_OK;
  k_soa_to_rows<<<nblocks(n), TPB, 0, s>>>(soa, rows, n, d, ld);
  count_launch();
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

int eval_target_soa(best_ctx* ctx, const double* theta, int64_t ld, int64_t n, double* logp,
                    double* grad, cudaStream_t s) {
  const bool mlp = ctx->tgt.has_mlp != 0;
  for (int64_t c0 = 0; c0 < n; c0 += kEvalChunk) {
    const int64_t m = (n - c0 < kEvalChunk) ? (n - c0) : kEvalChunk;
    if (mlp) {
      BEST_TRY(mlp_fp32_reserve(ctx, m < 1024 ? 1024 : m));
      k_prep_input<<<nblocks(m), TPB, 0, s>>>(theta + c0, ld, m, ctx->d, ctx->dp, ctx->X0);
      count_launch();
      BEST_TRY(mlp_fp32_run(ctx, m, grad != nullptr, s));
    }
    k_finish_target<<<nblocks(m), TPB, 0, s>>>(ctx->tgt, theta + c0, ld, m, ctx->mlp_out,
                                               ctx->mlp_grad, ctx->dp, logp + c0,
                                               grad ? grad + c0 : nullptr);
    count_launch();
  }
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

}  // namespace best
