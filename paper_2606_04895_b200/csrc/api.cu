// C-ABI entry points of libbest.so (include/best.h): argument checking, host-side setup
// (fp64 Cholesky of Sigma_inv, weight padding/upload), state management, dispatch.
#include <cmath>
#include <cstring>

#include "best_internal.h"
#include "tc_fused.h"

namespace best {

static thread_local std::string t_err;
void set_error(const std::string& msg) { t_err = msg; }
std::atomic<uint64_t> g_launches{0};

namespace {

bool chol_lower_host(const std::vector<double>& A, int d, std::vector<double>& Lo) {
  Lo.assign((size_t)d * d, 0.0);
  for (int j = 0; j < d; ++j) {
    double s = A[(size_t)j * d + j];
    for (int k = 0; k < j; ++k) s -= Lo[(size_t)j * d + k] * Lo[(size_t)j * d + k];
    if (!(s > 0.0) || !std::isfinite(s)) return false;
    const double ljj = std::sqrt(s);
    Lo[(size_t)j * d + j] = ljj;
    for (int i = j + 1; i < d; ++i) {
      double t = A[(size_t)i * d + j];
      for (int k = 0; k < j; ++k) t -= Lo[(size_t)i * d + k] * Lo[(size_t)j * d + k];
      Lo[(size_t)i * d + j] = t / ljj;
    }
  }
  return true;
}

}  // namespace
}  // namespace best

using namespace best;

extern "C" {

const char* best_last_error(void) { return t_err.c_str(); }
const char* best_version(void) { return "best-b200 0.2 (sm_100a)"; }
uint64_t best_launch_count(void) { return g_launches.load(); }

int best_create(const best_config* cfg, best_ctx** out) {
  if (!cfg || !out) { set_error("best_create: NULL argument"); return BEST_ERR_ARG; }
  *out = nullptr;
  const int d = cfg->d;
  if (d < 1 || d > kMaxD) { set_error("best_create: d must be in 1..32"); return BEST_ERR_ARG; }
  if (cfg->n_affine < 0 || cfg->n_affine > 16) { set_error("best_create: bad n_affine"); return BEST_ERR_ARG; }
  if (cfg->n_affine > 0) {
    if (!cfg->widths || !cfg->W_flat || !cfg->b_flat) { set_error("best_create: NULL MLP arrays"); return BEST_ERR_ARG; }
    if (cfg->widths[0] != d || cfg->widths[cfg->n_affine] != 1) {
      set_error("best_create: widths must start at d and end at 1");
      return BEST_ERR_ARG;
    }
    for (int k = 1; k < cfg->n_affine; ++k)
      if (cfg->widths[k] < 1 || cfg->widths[k] > 8192) { set_error("best_create: bad hidden width"); return BEST_ERR_ARG; }
  }
  if (cfg->activation != BEST_ACT_TANH && cfg->activation != BEST_ACT_SILU) {
    set_error("best_create: unknown activation");
    return BEST_ERR_ARG;
  }
  if (cfg->precision != BEST_PREC_FP32 && cfg->precision != BEST_PREC_BF16 && cfg->precision != BEST_PREC_FP32_TC) {
    set_error("best_create: unknown precision");
    return BEST_ERR_ARG;
  }
  if ((cfg->mu == nullptr) != (cfg->Sigma_inv == nullptr) || (cfg->lo == nullptr) != (cfg->hi == nullptr)) {
    set_error("best_create: mu/Sigma_inv and lo/hi come in pairs");
    return BEST_ERR_ARG;
  }
  if (cfg->banana_i >= 0 && (cfg->banana_i >= d || cfg->banana_j < 0 || cfg->banana_j >= d ||
                             cfg->banana_j == cfg->banana_i || !(cfg->banana_sigma > 0.f))) {
    set_error("best_create: bad banana indices / sigma");
    return BEST_ERR_ARG;
  }
  if (cfg->lo)
    for (int i = 0; i < d; ++i)
      if (!(cfg->hi[i] > cfg->lo[i])) { set_error("best_create: need hi > lo"); return BEST_ERR_ARG; }

  // host-side fp64 work
  std::vector<double> consts((size_t)5 * d * d, 0.0);  // mu | R | lo | hi | L (each d*d slot)
  double* h_mu = consts.data();
  double* h_R = h_mu + d * d;
  double* h_lo = h_R + d * d;
  double* h_hi = h_lo + d * d;
  double* h_L = h_hi + d * d;
  if (cfg->mu) {
    std::vector<double> P((size_t)d * d), Lp;
    for (int i = 0; i < d; ++i)
      for (int j = 0; j < d; ++j)
        P[(size_t)i * d + j] = 0.5 * (cfg->Sigma_inv[(size_t)i * d + j] + cfg->Sigma_inv[(size_t)j * d + i]);
    if (!chol_lower_host(P, d, Lp)) { set_error("best_create: Sigma_inv is not SPD"); return BEST_ERR_NOT_SPD; }
    for (int i = 0; i < d; ++i)
      for (int j = i; j < d; ++j) h_R[(size_t)i * d + j] = Lp[(size_t)j * d + i];  // R = Lp^T
    std::memcpy(h_mu, cfg->mu, sizeof(double) * d);
  }
  if (cfg->lo) {
    std::memcpy(h_lo, cfg->lo, sizeof(double) * d);
    std::memcpy(h_hi, cfg->hi, sizeof(double) * d);
  }
  for (int i = 0; i < d; ++i)
    for (int j = 0; j <= i; ++j) {
      const double v = cfg->L ? cfg->L[(size_t)i * d + j] : (i == j ? 1.0 : 0.0);
      if (i == j && !(v > 0.0)) { set_error("best_create: diag(L) must be positive"); return BEST_ERR_NOT_SPD; }
      h_L[(size_t)i * d + j] = v;
    }

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    set_error("best_create: no CUDA device (there is no CPU fallback)");
    return BEST_ERR_CUDA;
  }

  best_ctx* ctx = new best_ctx();
  ctx->d = d;
  ctx->dp = (d + 3) & ~3;
  ctx->n_affine = cfg->n_affine;
  ctx->activation = cfg->activation;
  ctx->precision = cfg->precision;
  auto fail = [&](int rc) { best_destroy(ctx); return rc; };

  int rc = dev_alloc(&ctx->dev_consts, consts.size());
  if (rc) return fail(rc);
  if (cudaMemcpy(ctx->dev_consts, consts.data(), sizeof(double) * consts.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
    set_error("best_create: upload failed");
    return fail(BEST_ERR_CUDA);
  }
  ctx->L_dev = ctx->dev_consts + 4 * d * d;
  if ((rc = dev_alloc(&ctx->Lraw_dev, (size_t)d * d + d))) return fail(rc);
  ctx->scale_dev = ctx->Lraw_dev + (size_t)d * d;
  {
    std::vector<double> ones((size_t)d, 1.0);
    if (cudaMemcpy(ctx->Lraw_dev, ctx->L_dev, sizeof(double) * d * d, cudaMemcpyDeviceToDevice) != cudaSuccess ||
        cudaMemcpy(ctx->scale_dev, ones.data(), sizeof(double) * d, cudaMemcpyHostToDevice) != cudaSuccess) {
      set_error("best_create: upload failed");
      return fail(BEST_ERR_CUDA);
    }
  }
  if ((rc = dev_alloc(&ctx->adapt_counts, 2))) return fail(rc);
  cudaMemset(ctx->adapt_counts, 0, sizeof(int64_t) * 2);

  TargetDev& T = ctx->tgt;
  T.d = d;
  T.has_gauss = cfg->mu ? 1 : 0;
  T.has_box = cfg->lo ? 1 : 0;
  T.mu = ctx->dev_consts;
  T.R = ctx->dev_consts + d * d;
  T.lo = ctx->dev_consts + 2 * d * d;
  T.hi = ctx->dev_consts + 3 * d * d;
  T.pen_kappa = cfg->pen_kappa;
  T.pen_gamma = cfg->pen_gamma;
  T.banana_i = cfg->banana_i;
  T.banana_j = cfg->banana_j;
  T.banana_sigma = cfg->banana_sigma;
  T.mlp_scale = cfg->mlp_scale;
  T.has_mlp = (cfg->n_affine > 0 && cfg->mlp_scale != 0.0f) ? 1 : 0;
  T.hard_box = 0;

  if (cfg->n_affine > 0) {
    ctx->widths.assign(cfg->widths, cfg->widths + cfg->n_affine + 1);
    ctx->wp.resize(cfg->n_affine + 1);
    for (int k = 0; k <= cfg->n_affine; ++k) ctx->wp[k] = (ctx->widths[k] + 3) & ~3;
    ctx->wp[cfg->n_affine] = 1;
    size_t wo = 0, bo = 0;
    for (int k = 0; k < cfg->n_affine; ++k) {
      const int nin = ctx->widths[k], nout = ctx->widths[k + 1];
      const int pin = ctx->wp[k], pout = ctx->wp[k + 1];
      std::vector<float> Wp((size_t)pin * pout, 0.f), bp(pout, 0.f);
      for (int r = 0; r < nout; ++r)
        for (int c = 0; c < nin; ++c) Wp[(size_t)r * pin + c] = cfg->W_flat[wo + (size_t)r * nin + c];
      for (int r = 0; r < nout; ++r) bp[r] = cfg->b_flat[bo + r];
      float *dW = nullptr, *db = nullptr;
      if ((rc = dev_alloc(&dW, Wp.size()))) return fail(rc);
      ctx->W.push_back(dW);
      if ((rc = dev_alloc(&db, bp.size()))) return fail(rc);
      ctx->b.push_back(db);
      cudaMemcpy(dW, Wp.data(), sizeof(float) * Wp.size(), cudaMemcpyHostToDevice);
      cudaMemcpy(db, bp.data(), sizeof(float) * bp.size(), cudaMemcpyHostToDevice);
      wo += (size_t)nin * nout;
      bo += nout;
    }
  }
  if (cfg->precision == BEST_PREC_BF16) {
    rc = tc_plan_create(ctx, cfg);
    if (rc) return fail(rc);
  } else if (cfg->precision == BEST_PREC_FP32_TC) {
    rc = tc32_plan_create(ctx, cfg);
    if (rc) return fail(rc);
  }
  if (cudaDeviceSynchronize() != cudaSuccess) { set_error("best_create: device error"); return fail(BEST_ERR_CUDA); }
  *out = ctx;
  return BEST_OK;
}

void best_destroy(best_ctx* ctx) {
  if (!ctx) return;
  if (ctx->tc) tc_plan_destroy(ctx);
  if (ctx->tc32) tc32_plan_destroy(ctx);
  for (auto p : ctx->W) cudaFree(p);
  for (auto p : ctx->b) cudaFree(p);
  for (auto p : ctx->H) cudaFree(p);
  for (auto p : ctx->Dact) cudaFree(p);
  cudaFree(ctx->X0); cudaFree(ctx->delta[0]); cudaFree(ctx->delta[1]);
  cudaFree(ctx->mlp_out); cudaFree(ctx->mlp_grad);
  cudaFree(ctx->dev_consts); cudaFree(ctx->adapt_counts); cudaFree(ctx->Lraw_dev); cudaFree(ctx->lg_scratch);
  delete ctx;
}

}  // extern "C"
