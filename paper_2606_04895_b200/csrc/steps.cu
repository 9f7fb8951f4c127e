// Exact-path step kernels: MH (A4), MALA (A5), HMC (A6), AIES (A7), accept/trace/counters (A8).
// One thread per chain, fp64, SoA state [d][B].  Each kernel is one half of a step (propose /
// accept) with the emulator passes (emulator_fp32.cu) in between.
#include "best_internal.h"
#include "device_math.cuh"
#include "gram.cuh"

namespace best {
namespace {

constexpr int TPB = 128;
inline int nblocks(int64_t n) { return (int)((n + TPB - 1) / TPB); }

struct Chains {  // device pointers of one best_state
  int64_t B;
  int d;
  uint32_t chain0;  // Philox chain id of chain 0
  double *theta, *grad, *logp, *p_theta, *p_grad, *p_logp, *q, *h0, *last_la;
  unsigned long long* n_accept;
};

__device__ __forceinline__ void load_col(const double* a, int64_t ld, int64_t c, int d, double* v) {
  for (int i = 0; i < d; ++i) v[i] = a[i * ld + c];
}
__device__ __forceinline__ void store_col(double* a, int64_t ld, int64_t c, int d, const double* v) {
  for (int i = 0; i < d; ++i) a[i * ld + c] = v[i];
}

// ---- MH: theta' = theta + eps L xi -----------------------------------------------------------
__global__ void k_mh_propose(Chains S, const double* __restrict__ L, uint64_t seed, uint64_t step,
                             double eps) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= S.B) return;
  const int d = S.d;
  double xi[kMaxD], dx[kMaxD];
  draw_normals<double>(seed, S.chain0 + (uint32_t)c, step, d, xi);
  for (int i = 0; i < d; ++i) xi[i] *= eps;
  tri_L_apply<double>(L, d, xi, dx);
  for (int i = 0; i < d; ++i) S.p_theta[i * S.B + c] = S.theta[i * S.B + c] + dx[i];
}

__global__ void k_mh_accept(Chains S, uint64_t seed, uint64_t step) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= S.B) return;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)c, step, 0u, seed);
  const double la = S.p_logp[c] - S.logp[c];
  S.last_la[c] = la;
  if (accept_rule<double>(u01<double>(w.x), la)) {
    for (int i = 0; i < S.d; ++i) S.theta[i * S.B + c] = S.p_theta[i * S.B + c];
    S.logp[c] = S.p_logp[c];
    S.n_accept[c] += 1ull;
  }
}

// ---- MALA: z' = z + eps g_z + sqrt(2 eps) xi  (eq 2.3) -----------------------------------------
__global__ void k_mala_propose(Chains S, const double* __restrict__ L, uint64_t seed, uint64_t step,
                               double eps) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= S.B) return;
  const int d = S.d;
  double xi[kMaxD], g[kMaxD], gz[kMaxD], dx[kMaxD];
  draw_normals<double>(seed, S.chain0 + (uint32_t)c, step, d, xi);
  load_col(S.grad, S.B, c, d, g);
  tri_Lt_apply<double>(L, d, g, gz);
  const double sq = sqrt(2.0 * eps);
  for (int i = 0; i < d; ++i) gz[i] = eps * gz[i] + sq * xi[i];
  tri_L_apply<double>(L, d, gz, dx);
  for (int i = 0; i < d; ++i) S.p_theta[i * S.B + c] = S.theta[i * S.B + c] + dx[i];
}

__global__ void k_mala_accept(Chains S, const double* __restrict__ L, uint64_t seed, uint64_t step,
                              double eps) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= S.B) return;
  const int d = S.d;
  double xi[kMaxD], g[kMaxD], gz[kMaxD], gzp[kMaxD];
  draw_normals<double>(seed, S.chain0 + (uint32_t)c, step, d, xi);
  load_col(S.grad, S.B, c, d, g);
  tri_Lt_apply<double>(L, d, g, gz);
  load_col(S.p_grad, S.B, c, d, g);
  tri_Lt_apply<double>(L, d, g, gzp);
  const double sq = sqrt(2.0 * eps);
  double fwd = 0.0, bwd = 0.0;
  for (int i = 0; i < d; ++i) {
    const double f = sq * xi[i];
    const double r = -(eps * (gz[i] + gzp[i]) + sq * xi[i]);
    fwd += f * f;
    bwd += r * r;
  }
  const double la = S.p_logp[c] - S.logp[c] + (-bwd / (4.0 * eps)) - (-fwd / (4.0 * eps));
  S.last_la[c] = la;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)c, step, 0u, seed);
  if (accept_rule<double>(u01<double>(w.x), la)) {
    for (int i = 0; i < d; ++i) {
      S.theta[i * S.B + c] = S.p_theta[i * S.B + c];
      S.grad[i * S.B + c] = g[i];
    }
    S.logp[c] = S.p_logp[c];
    S.n_accept[c] += 1ull;
  }
}

// ---- HMC: kick-drift-kick leapfrog in whitened space (eq 2.1 / 2.8) ----------------------------
__global__ void k_hmc_begin(Chains S, const double* __restrict__ L, uint64_t seed, uint64_t step,
                            double eps) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= S.B) return;
  const int d = S.d;
  double q[kMaxD], g[kMaxD], gz[kMaxD], dx[kMaxD];
  draw_normals<double>(seed, S.chain0 + (uint32_t)c, step, d, q);
  double kin = 0.0;
  for (int i = 0; i < d; ++i) kin += q[i] * q[i];
  S.h0[c] = -S.logp[c] + 0.5 * kin;
  load_col(S.grad, S.B, c, d, g);
  tri_Lt_apply<double>(L, d, g, gz);
  for (int i = 0; i < d; ++i) q[i] += 0.5 * eps * gz[i];
  store_col(S.q, S.B, c, d, q);
  for (int i = 0; i < d; ++i) gz[i] = eps * q[i];
  tri_L_apply<double>(L, d, gz, dx);
  for (int i = 0; i < d; ++i) S.p_theta[i * S.B + c] = S.theta[i * S.B + c] + dx[i];
}

// after the gradient at the l-th drift position: kick, then either drift again or accept
__global__ void k_hmc_kick(Chains S, const double* __restrict__ L, uint64_t seed, uint64_t step,
                           double eps, int last) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= S.B) return;
  const int d = S.d;
  double q[kMaxD], g[kMaxD], gz[kMaxD], dx[kMaxD];
  load_col(S.q, S.B, c, d, q);
  load_col(S.p_grad, S.B, c, d, g);
  tri_Lt_apply<double>(L, d, g, gz);
  const double cc = last ? 0.5 * eps : eps;
  for (int i = 0; i < d; ++i) q[i] += cc * gz[i];
  if (!last) {
    store_col(S.q, S.B, c, d, q);
    for (int i = 0; i < d; ++i) gz[i] = eps * q[i];
    tri_L_apply<double>(L, d, gz, dx);
    for (int i = 0; i < d; ++i) S.p_theta[i * S.B + c] += dx[i];
    return;
  }
  double kin = 0.0;
  for (int i = 0; i < d; ++i) kin += q[i] * q[i];
  const double H1 = -S.p_logp[c] + 0.5 * kin;
  const double la = S.h0[c] - H1;
  S.last_la[c] = la;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)c, step, 0u, seed);
  if (accept_rule<double>(u01<double>(w.x), la)) {
    for (int i = 0; i < d; ++i) {
      S.theta[i * S.B + c] = S.p_theta[i * S.B + c];
      S.grad[i * S.B + c] = g[i];
    }
    S.logp[c] = S.p_logp[c];
    S.n_accept[c] += 1ull;
  }
}

// ---- AIES stretch move, one half-ensemble (eq 2.13-2.15) ---------------------------------------
// (`half` walkers are updated by this launch; partners come from the `n_oth` walkers of the other half: the
// same number unless the ensemble is sharded over ranks, best_set_aies_exchange)
__global__ void k_aies_propose(Chains S, uint64_t seed, uint64_t step, double a, int64_t own0,
                               int64_t oth0, int64_t half, int64_t n_oth) {
  const int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (r >= half) return;
  const int64_t i = own0 + r;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)i, step, 0u, seed);
  const int64_t j = oth0 + (int64_t)__umulhi(w.z, (uint32_t)n_oth);
  const double t = u01<double>(w.y) * (a - 1.0) + 1.0;
  const double z = t * t / a;
  for (int k = 0; k < S.d; ++k) {
    const double xi = S.theta[k * S.B + i], xj = S.theta[k * S.B + j];
    S.p_theta[k * S.B + r] = xj + z * (xi - xj);
  }
}

__global__ void k_aies_accept(Chains S, uint64_t seed, uint64_t step, double a, int64_t own0,
                              int64_t half) {
  const int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (r >= half) return;
  const int64_t i = own0 + r;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)i, step, 0u, seed);
  const double t = u01<double>(w.y) * (a - 1.0) + 1.0;
  const double z = t * t / a;
  const double la = (double)(S.d - 1) * log(z) + S.p_logp[r] - S.logp[i];
  S.last_la[i] = la;
  if (accept_rule<double>(u01<double>(w.x), la)) {
    for (int k = 0; k < S.d; ++k) S.theta[k * S.B + i] = S.p_theta[k * S.B + r];
    S.logp[i] = S.p_logp[r];
    S.n_accept[i] += 1ull;
  }
}

// Differential-evolution move, eq (2.16) (reading R23): x' = x_i + gamma (x_j - x_k),
// j != k from the other half (control words 2 and 3), gamma = (1 + sigma * n0) 2.38 / sqrt(2 d) with n0
// the first normal of slot 1; symmetric proposal, log alpha = log pi(x') - log pi(x_i).
__global__ void k_de_propose(Chains S, uint64_t seed, uint64_t step, double sigma, int64_t own0,
                             int64_t oth0, int64_t half, int64_t n_oth) {
  const int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (r >= half) return;
  const int64_t i = own0 + r;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)i, step, 0u, seed);
  const int64_t jr = (int64_t)__umulhi(w.z, (uint32_t)n_oth);
  int64_t kr = (int64_t)__umulhi(w.w, (uint32_t)(n_oth - 1));
  if (kr >= jr) kr += 1;
  const uint4 wn = philox4x32_10(S.chain0 + (uint32_t)i, step, 1u, seed);
  double n0, n1;
  box_muller(wn.x, wn.y, n0, n1);
  const double gamma = (1.0 + sigma * n0) * (2.38 / sqrt(2.0 * (double)S.d));
  const int64_t j = oth0 + jr, k = oth0 + kr;
  for (int q = 0; q < S.d; ++q)
    S.p_theta[q * S.B + r] = S.theta[q * S.B + i] + gamma * (S.theta[q * S.B + j] - S.theta[q * S.B + k]);
}

__global__ void k_de_accept(Chains S, uint64_t seed, uint64_t step, int64_t own0, int64_t half) {
  const int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (r >= half) return;
  const int64_t i = own0 + r;
  const uint4 w = philox4x32_10(S.chain0 + (uint32_t)i, step, 0u, seed);
  const double la = S.p_logp[r] - S.logp[i];
  S.last_la[i] = la;
  if (accept_rule<double>(u01<double>(w.x), la)) {
    for (int q = 0; q < S.d; ++q) S.theta[q * S.B + i] = S.p_theta[q * S.B + r];
    S.logp[i] = S.p_logp[r];
    S.n_accept[i] += 1ull;
  }
}

__global__ void k_trace(const double* __restrict__ theta, int64_t B, int d, float* __restrict__ out) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= B) return;
  for (int i = 0; i < d; ++i) out[c * d + i] = (float)theta[i * B + c];
}

// ---- A9: running covariance, deterministic per-block partial sums ------------------------------
constexpr int COV_TPB = 128;  // d*COV_TPB doubles of dynamic smem: 32 KB at d = 32
// acc[blk][e]: e = 0 count, 1..d sums of (theta - ref), then d*d sums of products
__global__ void __launch_bounds__(COV_TPB)
k_cov_accumulate(const double* __restrict__ theta, int64_t B, int d, const double* __restrict__ ref,
                 double* __restrict__ acc) {
  extern __shared__ double xs[];  // [d][COV_TPB]
  const int64_t c0 = blockIdx.x * (int64_t)COV_TPB;
  const int64_t c = c0 + threadIdx.x;
  const int nvalid = (int)((B - c0 < COV_TPB) ? (B - c0) : COV_TPB);
  for (int i = 0; i < d; ++i)
    xs[i * COV_TPB + threadIdx.x] = (c < B) ? theta[i * B + c] - ref[i] : 0.0;
  __syncthreads();
  const int ne = 1 + d + d * d;
  double* mine = acc + (size_t)blockIdx.x * ne;
  for (int e = threadIdx.x; e < ne; e += COV_TPB) {
    double s = 0.0;
    if (e == 0) {
      s = (double)nvalid;
    } else if (e <= d) {
      const double* x = xs + (e - 1) * COV_TPB;
      for (int t = 0; t < nvalid; ++t) s += x[t];
    } else {
      const int i = (e - 1 - d) / d, j = (e - 1 - d) % d;
      const double *x = xs + i * COV_TPB, *y = xs + j * COV_TPB;
      for (int t = 0; t < nvalid; ++t) s += x[t] * y[t];
    }
    mine[e] += s;
  }
}

// C = scatter/(n-1), C_ii *= (1+jitter), L = chol(C) with jitter x10 retries; swap L on success.
__global__ void k_cov_finalize(double* __restrict__ acc, int nblk, int d, double jitter,
                               double* __restrict__ L, double* __restrict__ Lraw,
                               const double* __restrict__ scale, long long* __restrict__ counts) {
  __shared__ double S[1 + kMaxD + kMaxD * kMaxD];
  __shared__ double Cm[kMaxD * kMaxD], Lt[kMaxD * kMaxD];
  const int ne = 1 + d + d * d;
  for (int e = threadIdx.x; e < ne; e += blockDim.x) {   // partials are added in block order (fixed), loads 8 at a time
    double s = 0.0;
    int b = 0;
    for (; b + 8 <= nblk; b += 8) {
      double v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = acc[(size_t)(b + u) * ne + e];
#pragma unroll
      for (int u = 0; u < 8; ++u) s += v[u];
    }
    for (; b < nblk; ++b) s += acc[(size_t)b * ne + e];
    S[e] = s;
    for (b = 0; b < nblk; ++b) acc[(size_t)b * ne + e] = 0.0;   // the next window starts from zero
  }
  __syncthreads();
  if (threadIdx.x != 0) return;
  const double n = S[0];
  bool ok = false;
  if (n >= 2.0) {
    double jit = jitter;
    for (int attempt = 0; attempt < 6 && !ok; ++attempt) {
      for (int i = 0; i < d; ++i)
        for (int j = 0; j < d; ++j) {
          const double sij = 0.5 * (S[1 + d + i * d + j] + S[1 + d + j * d + i]);
          Cm[i * d + j] = (sij - S[1 + i] * S[1 + j] / n) / (n - 1.0);
        }
      for (int i = 0; i < d; ++i) Cm[i * d + i] *= (1.0 + jit);
      ok = true;
      for (int j = 0; j < d && ok; ++j) {
        double s = Cm[j * d + j];
        for (int k = 0; k < j; ++k) s -= Lt[j * d + k] * Lt[j * d + k];
        if (!(s > 0.0)) { ok = false; break; }
        const double ljj = sqrt(s);
        Lt[j * d + j] = ljj;
        for (int i = j + 1; i < d; ++i) {
          double t = Cm[i * d + j];
          for (int k = 0; k < j; ++k) t -= Lt[i * d + k] * Lt[j * d + k];
          Lt[i * d + j] = t / ljj;
        }
      }
      jit *= 10.0;
    }
  }
  if (ok) {
    for (int i = 0; i < d; ++i)
      for (int j = 0; j < d; ++j) {
        const double v = (j <= i) ? Lt[i * d + j] : 0.0;
        Lraw[i * d + j] = v;
        L[i * d + j] = v * scale[j];   // per-dimension step factors (8(f)#1) survive the update
      }
    counts[0] += 1;
  } else {
    counts[1] += 1;
  }
}

// ---- A9 across ranks ("covariance adaptation = one all-reduce of d^2+d+1 fp64 values per window") ----
// Every rank's window sums are taken about its OWN reference point, so a rank's packet carries that point as well:
// packet = [ n | ref (d) | S1 = sum(theta - ref) (d) | S2 = sum (theta - ref)(theta - ref)^T (d*d) ].
// k_cov_pack adds the per-block partials in block order (as k_cov_finalize does) and clears them.
__global__ void k_cov_pack(double* __restrict__ acc, int nblk, int d, const double* __restrict__ ref,
                           double* __restrict__ packet) {
  const int ne = 1 + d + d * d;
  for (int e = threadIdx.x; e < ne; e += blockDim.x) {
    double s = 0.0;
    for (int b = 0; b < nblk; ++b) { s += acc[(size_t)b * ne + e]; acc[(size_t)b * ne + e] = 0.0; }
    packet[e == 0 ? 0 : e + d] = s;
  }
  for (int i = threadIdx.x; i < d; i += blockDim.x) packet[1 + i] = ref[i];
}
// The gathered packets, rank 0 first, moved to rank 0's reference point and added in rank order (every rank gets
// the same bits): with delta = ref_k - ref_0, theta - ref_0 = (theta - ref_k) + delta, hence
//   S1' = S1 + n delta,   S2'_ij = S2_ij + S1_i delta_j + delta_i S1_j + n delta_i delta_j.
// The total goes to partial block 0 (the others are zero after k_cov_pack): k_cov_finalize then runs unchanged.
__global__ void k_cov_combine(const double* __restrict__ gathered, int world, int d, double* __restrict__ acc) {
  const int ne = 1 + d + d * d, np = 1 + 2 * d + d * d;
  for (int e = threadIdx.x; e < ne; e += blockDim.x) {
    double tot = 0.0;
    for (int k = 0; k < world; ++k) {
      const double* pk = gathered + (size_t)k * np;
      const double n = pk[0];
      const double *rk = pk + 1, *r0 = gathered + 1, *s1 = pk + 1 + d, *s2 = pk + 1 + 2 * d;
      if (e == 0) {
        tot += n;
      } else if (e <= d) {
        const int i = e - 1;
        tot += s1[i] + n * (rk[i] - r0[i]);
      } else {
        const int i = (e - 1 - d) / d, j = (e - 1 - d) % d;
        const double di = rk[i] - r0[i], dj = rk[j] - r0[j];
        tot += s2[i * d + j] + s1[i] * dj + di * s1[j] + n * di * dj;
      }
    }
    acc[e] = tot;
  }
}

Chains chains_of(best_state* st) {
  Chains S;
  S.B = st->B; S.d = st->ctx->d; S.chain0 = (uint32_t)st->chain0;
  S.theta = st->theta; S.grad = st->grad; S.logp = st->logp;
  S.p_theta = st->p_theta; S.p_grad = st->p_grad; S.p_logp = st->p_logp;
  S.q = st->q; S.h0 = st->h0; S.last_la = st->last_la; S.n_accept = st->n_accept;
  return S;
}

}  // namespace

static int close_window(best_ctx* ctx, best_state* st, cudaStream_t s) {
  if (st->xchg_fn) {
    // own sums -> packet -> the caller's all-gather (enqueued on `s`) -> all ranks' sums about rank 0's reference
    const int d = ctx->d;
    const int64_t np = 1 + 2 * (int64_t)d + (int64_t)d * d;
    k_cov_pack<<<1, 1024, 0, s>>>(st->cov_acc, st->cov_blocks, d, st->cov_ref, st->xchg_buf);
    count_launch();
    BEST_CUDA(cudaGetLastError());
    const int rc = st->xchg_fn(st->xchg_buf, st->xchg_buf + np, np, (void*)s, st->xchg_user);
    if (rc != 0) { set_error("best_set_adaptation_exchange: the exchange callback returned an error"); return BEST_ERR_CUDA; }
    k_cov_combine<<<1, 1024, 0, s>>>(st->xchg_buf + np, st->xchg_world, d, st->cov_acc);
    count_launch();
    BEST_CUDA(cudaGetLastError());
  }
  k_cov_finalize<<<1, 1024, 0, s>>>(st->cov_acc, st->cov_blocks, ctx->d, st->jitter, ctx->L_dev, ctx->Lraw_dev,
                                   ctx->scale_dev, (long long*)ctx->adapt_counts);
  count_launch();
  st->win_steps = 0;
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

int after_step(best_ctx* ctx, best_state* st, int64_t t, float* trace, int thin, bool adapt,
               cudaStream_t s) {
  if (trace && thin > 0 && (t + 1) % thin == 0) {
    const int64_t slot = (t + 1) / thin - 1;
    k_trace<<<nblocks(st->B), TPB, 0, s>>>(st->theta, st->B, ctx->d,
                                           trace + (size_t)slot * st->B * ctx->d);
    count_launch();
  }
  if (adapt && st->adapt_every > 0) {
    const int nblk = (int)((st->B + COV_TPB - 1) / COV_TPB);   // <= st->cov_blocks (adapt_reset)
    k_cov_accumulate<<<nblk, COV_TPB, sizeof(double) * ctx->d * COV_TPB, s>>>(
        st->theta, st->B, ctx->d, st->cov_ref, st->cov_acc);
    count_launch();
    if (++st->win_steps >= st->adapt_every) BEST_TRY(close_window(ctx, st, s));
  }
  return BEST_OK;
}

int adapt_acquire_buffer(best_state* st, cudaStream_t s, int* buf) {
  const int b = st->win_flip;
  st->win_flip ^= 1;
  BEST_CUDA(cudaStreamWaitEvent(s, st->ev_gram[b], 0));   // (never recorded: no-op)
  *buf = b;
  return BEST_OK;
}

// Called right after the persistent launch of a segment on `s`.  The Gram kernel runs on the state's side stream
// behind that launch, so it overlaps the NEXT segment's persistent kernel (it fits on the SMs that kernel leaves
// idle: 20 of 148 at 16 384 chains, the tail of the last wave otherwise); Gram launches are ordered among
// themselves by the side stream, the window close waits for the last one on `s`.
int adapt_window_rows(best_ctx* ctx, best_state* st, int buf, int64_t n_steps, cudaStream_t s) {
  const int d = ctx->d;
  BEST_CUDA(cudaEventRecord(st->ev_seg[buf], s));
  BEST_CUDA(cudaStreamWaitEvent(st->side, st->ev_seg[buf], 0));
  k_gram_window<<<st->cov_blocks / 2, G_TPB, 0, st->side>>>(st->win_buf[buf], st->win_steps * st->B, n_steps * st->B, d,
                                                            st->cov_ref, st->cov_acc);
  count_launch();
  BEST_CUDA(cudaGetLastError());
  BEST_CUDA(cudaEventRecord(st->ev_gram[buf], st->side));
  st->win_steps += n_steps;
  if (st->win_steps >= st->adapt_every) {
    BEST_CUDA(cudaStreamWaitEvent(s, st->ev_gram[buf], 0));
    BEST_TRY(close_window(ctx, st, s));
  }
  return BEST_OK;
}

void adapt_free(best_state* st) {
  if (st->side) cudaStreamSynchronize(st->side);
  cudaFree(st->cov_acc); cudaFree(st->cov_ref); cudaFree(st->win_buf[0]); cudaFree(st->win_buf[1]);
  cudaFree(st->xchg_buf); st->xchg_buf = nullptr; st->xchg_fn = nullptr;
  cudaFree(st->aies_buf); st->aies_buf = nullptr; st->aies_fn = nullptr;
  for (int i = 0; i < 2; ++i) {
    if (st->ev_seg[i]) cudaEventDestroy(st->ev_seg[i]);
    if (st->ev_gram[i]) cudaEventDestroy(st->ev_gram[i]);
    st->ev_seg[i] = st->ev_gram[i] = nullptr;
  }
  if (st->side) cudaStreamDestroy(st->side);
  st->side = nullptr;
  st->cov_acc = nullptr; st->cov_ref = nullptr; st->win_buf[0] = st->win_buf[1] = nullptr;
  st->cov_blocks = 0; st->win_cap_steps = 0;
}

// Opens a fresh window for `st`: zeroed per-block sums, shift = chain 0's current position (any fixed
// reference removes the large mean^2 term), and on the tensor path the window buffer the persistent kernel
// writes its post-accept states to (at most 256 MB: longer windows are fed to the Gram kernel in segments).
int adapt_reset(best_ctx* ctx, best_state* st, cudaStream_t s) {
  const int d = ctx->d;
  const size_t ne = 1 + d + (size_t)d * d;
  int nblk;
  int64_t cap = 0;
  if (ctx->precision == BEST_PREC_BF16) {
    cap = (int64_t)((128ull << 20) / ((size_t)st->B * d * sizeof(float)));   // two buffers of at most 128 MB
    cap = cap < 1 ? 1 : (cap > st->adapt_every ? st->adapt_every : cap);
    // grid of the window's Gram kernel: one CTA per 64-row tile up to four per SM, fixed for the whole window
    // (with the window length and B it determines the summation order); two partial sets (row parity) per CTA
    const int64_t tiles = (st->B * (int64_t)st->adapt_every + G_ROWS - 1) / G_ROWS;
    const int64_t want = (tiles + 15) / 16;   // >= 16 tiles per CTA before the grid grows: few partial sets for small batches
    nblk = 2 * (int)(want < 1 ? 1 : (want < 592 ? want : 592));
  } else {
    nblk = (int)((st->B + COV_TPB - 1) / COV_TPB);
  }
  if (nblk > st->cov_blocks) {
    cudaFree(st->cov_acc);
    st->cov_acc = nullptr; st->cov_blocks = 0;
    BEST_TRY(dev_alloc(&st->cov_acc, ne * nblk));
    st->cov_blocks = nblk;
  }
  if (!st->cov_ref) BEST_TRY(dev_alloc(&st->cov_ref, (size_t)d));
  if (cap > 0) {
    if (!st->side) {
      BEST_CUDA(cudaStreamCreateWithFlags(&st->side, cudaStreamNonBlocking));
      for (int i = 0; i < 2; ++i) {
        BEST_CUDA(cudaEventCreateWithFlags(&st->ev_seg[i], cudaEventDisableTiming));
        BEST_CUDA(cudaEventCreateWithFlags(&st->ev_gram[i], cudaEventDisableTiming));
      }
    }
    BEST_CUDA(cudaStreamSynchronize(st->side));
    if (cap > st->win_cap_alloc) {
      for (int i = 0; i < 2; ++i) {
        cudaFree(st->win_buf[i]);
        st->win_buf[i] = nullptr;
      }
      st->win_cap_alloc = 0;
      for (int i = 0; i < 2; ++i) BEST_TRY(dev_alloc(&st->win_buf[i], (size_t)cap * st->B * d));
      st->win_cap_alloc = cap;
    }
    st->win_cap_steps = cap;
  }
  BEST_CUDA(cudaMemsetAsync(st->cov_acc, 0, sizeof(double) * ne * st->cov_blocks, s));
  BEST_CUDA(cudaMemcpy2DAsync(st->cov_ref, sizeof(double), st->theta, sizeof(double) * st->B, sizeof(double), d,
                              cudaMemcpyDeviceToDevice, s));
  st->win_steps = 0;
  return BEST_OK;
}

int step_mh(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, double eps, float* trace,
            int thin, cudaStream_t s) {
  Chains S = chains_of(st);
  const int nb = nblocks(st->B);
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = st->step + (uint64_t)t;
    k_mh_propose<<<nb, TPB, 0, s>>>(S, ctx->L_dev, seed, step, eps);
    count_launch();
    BEST_TRY(eval_target_soa(ctx, st->p_theta, st->B, st->B, st->p_logp, nullptr, s));
    k_mh_accept<<<nb, TPB, 0, s>>>(S, seed, step);
    count_launch();
    BEST_TRY(after_step(ctx, st, t, trace, thin, true, s));
  }
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

int step_mala(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, double eps,
              float* trace, int thin, cudaStream_t s) {
  Chains S = chains_of(st);
  const int nb = nblocks(st->B);
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = st->step + (uint64_t)t;
    k_mala_propose<<<nb, TPB, 0, s>>>(S, ctx->L_dev, seed, step, eps);
    count_launch();
    BEST_TRY(eval_target_soa(ctx, st->p_theta, st->B, st->B, st->p_logp, st->p_grad, s));
    k_mala_accept<<<nb, TPB, 0, s>>>(S, ctx->L_dev, seed, step, eps);
    count_launch();
    BEST_TRY(after_step(ctx, st, t, trace, thin, true, s));
  }
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

int step_hmc(best_ctx* ctx, best_state* st, int64_t n_traj, uint64_t seed, double eps, int n_leapfrog,
             float* trace, int thin, cudaStream_t s) {
  Chains S = chains_of(st);
  const int nb = nblocks(st->B);
  for (int64_t t = 0; t < n_traj; ++t) {
    const uint64_t step = st->step + (uint64_t)t;
    k_hmc_begin<<<nb, TPB, 0, s>>>(S, ctx->L_dev, seed, step, eps);
    count_launch();
    for (int l = 1; l <= n_leapfrog; ++l) {
      BEST_TRY(eval_target_soa(ctx, st->p_theta, st->B, st->B, st->p_logp, st->p_grad, s));
      k_hmc_kick<<<nb, TPB, 0, s>>>(S, ctx->L_dev, seed, step, eps, l == n_leapfrog ? 1 : 0);
      count_launch();
    }
    BEST_TRY(after_step(ctx, st, t, trace, thin, true, s));
  }
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

// ---- sharded ensemble moves ("AIES = one all-gather of the complementary half's positions per
// half-step"): the slice this rank has just updated, theta rows then log pi, [d + 1][cnt] ----------------------
__global__ void k_aies_pack(const double* __restrict__ theta, const double* __restrict__ logp, int64_t B, int d,
                            int64_t first, int64_t cnt, double* __restrict__ send) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= cnt) return;
  for (int k = 0; k < d; ++k) send[(int64_t)k * cnt + c] = theta[(int64_t)k * B + first + c];
  send[(int64_t)d * cnt + c] = logp[first + c];
}
__global__ void k_aies_unpack(const double* __restrict__ recv, int world, int d, int64_t cnt, int64_t half0,
                              double* __restrict__ theta, double* __restrict__ logp, int64_t B) {
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;   // walker of the half: rank c / cnt, slot c % cnt
  if (c >= cnt * world) return;
  const double* src = recv + (c / cnt) * (int64_t)(d + 1) * cnt + (c % cnt);
  for (int k = 0; k < d; ++k) theta[(int64_t)k * B + half0 + c] = src[(int64_t)k * cnt];
  logp[half0 + c] = src[(int64_t)d * cnt];
}

int aies_exchange(best_ctx* ctx, best_state* st, int64_t half0, cudaStream_t s) {
  const int d = ctx->d;
  const int64_t cnt = st->B / 2 / st->aies_world, n = (int64_t)(d + 1) * cnt;
  k_aies_pack<<<nblocks(cnt), TPB, 0, s>>>(st->theta, st->logp, st->B, d, half0 + st->aies_rank * cnt, cnt, st->aies_buf);
  count_launch();
  BEST_CUDA(cudaGetLastError());
  if (st->aies_fn(st->aies_buf, st->aies_buf + n, n, (void*)s, st->aies_user) != 0) {
    set_error("best_set_aies_exchange: the exchange callback returned an error");
    return BEST_ERR_CUDA;
  }
  k_aies_unpack<<<nblocks(cnt * st->aies_world), TPB, 0, s>>>(st->aies_buf + n, st->aies_world, d, cnt, half0, st->theta,
                                                           st->logp, st->B);
  count_launch();
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

int step_aies(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, double a, float* trace,
              int thin, cudaStream_t s, bool de) {
  Chains S = chains_of(st);
  const int64_t half = st->B / 2;
  // sharded: this rank moves `cnt` walkers of each half, partners are drawn from the whole other half
  const int64_t cnt = st->aies_fn ? half / st->aies_world : half, off = st->aies_fn ? st->aies_rank * cnt : 0;
  const int nb = nblocks(cnt);
  for (int64_t t = 0; t < n_steps; ++t) {
    const uint64_t step = st->step + (uint64_t)t;
    for (int hh = 0; hh < 2; ++hh) {
      const int64_t half0 = hh == 0 ? 0 : half, own0 = half0 + off, oth0 = hh == 0 ? half : 0;
      if (de) k_de_propose<<<nb, TPB, 0, s>>>(S, seed, step, a, own0, oth0, cnt, half);   // a = sigma_gamma
      else k_aies_propose<<<nb, TPB, 0, s>>>(S, seed, step, a, own0, oth0, cnt, half);
      count_launch();
      BEST_TRY(eval_target_soa(ctx, st->p_theta, st->B, cnt, st->p_logp, nullptr, s));
      if (de) k_de_accept<<<nb, TPB, 0, s>>>(S, seed, step, own0, cnt);
      else k_aies_accept<<<nb, TPB, 0, s>>>(S, seed, step, a, own0, cnt);
      count_launch();
      if (st->aies_fn) BEST_TRY(aies_exchange(ctx, st, half0, s));
    }
    BEST_TRY(after_step(ctx, st, t, trace, thin, false, s));
  }
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

}  // namespace best
