/* best.h — C-ABI boundary of the B200-native hot path of BEST
 * ("Posterior sampling in the Age of Emulators", arxiv/paper_2606_04895; PAPER.md = "P").
 *
 * What sits behind it (SURVEY.md §8(a), rows A1–A9): many MCMC chains advanced in lockstep on one
 * GPU, every step evaluating a differentiable MLP log-likelihood emulator and its θ-gradient for
 * the whole chain batch (P:L7, L38, L147-149).  The interface follows the paper's statement of the
 * problem: target + bounds at construction, method / n_steps / n_chains at sampling,
 * acceptance counters / evaluations / samples / covariance out.
 *
 * Conventions
 *  - Every function returns BEST_OK (0) or a negative error code; nothing throws.  The text of
 *    the last error on the calling thread is returned by best_last_error().
 *  - "host" pointers are ordinary CPU memory, "dev" pointers are CUDA device memory on the
 *    current device, "host|dev" means either (detected with cudaPointerGetAttributes).
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Kernels are
 *    enqueued on it and the call returns without waiting, unless stated otherwise; calls that
 *    take host output buffers synchronise the stream before returning.
 *  - best_create / best_state_create deep-copy their inputs; the caller keeps its arrays.
 *  - θ, log π and ∇θ log π at this boundary are in the ORIGINAL (unwhitened) space and log π is
 *    unnormalised: the constant log|det L| of eq (2.12) is NOT added — it cancels in
 *    every accept ratio.
 *  - There is no CPU fallback and no other backend: without a CUDA device every compute entry
 *    point returns BEST_ERR_CUDA.
 *  - Concurrency: a context and ALL its states share emulator scratch (activation derivatives, exact-path
 *    layer buffers) and the whitening factor, so a context is driven from ONE stream (and one host thread) at
 *    a time; different contexts are independent.  Calls documented as "synchronises the device" order
 *    themselves against work in flight on any stream.
 *  - Environment: BEST_TC_ROWS = 128 | 256 | 265 | 233 | 264 | 232 | 64 | 32, read at best_create, forces a tile
 *    geometry of the tensor-core path that the widths allow (tests compare geometries bit for bit); results
 *    do not depend on it.  No other environment variable is read.
 */
#ifndef BEST_H_
#define BEST_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct best_ctx best_ctx;     /* opaque: device copies of weights, R, L, box, scratch */
typedef struct best_state best_state; /* opaque: chain state on the device                    */

enum {
  BEST_OK = 0,
  BEST_ERR_ARG = -1,         /* bad argument (NULL, size, eps <= 0, odd walker count, a <= 1 …) */
  BEST_ERR_CUDA = -2,        /* CUDA runtime error / no device                                   */
  BEST_ERR_NOT_SPD = -3,     /* Sigma_inv not SPD, or diag(L) not positive                       */
  BEST_ERR_UNSUPPORTED = -4, /* shape not supported by the requested precision path              */
  BEST_ERR_ALLOC = -5
};
enum { BEST_ACT_TANH = 0, BEST_ACT_SILU = 1 };
enum {
  BEST_PREC_FP32 = 0, /* FFMA emulator, fp64 chain state and Gaussian/whitening algebra          */
  BEST_PREC_BF16 = 1, /* tcgen05 tensor-core emulator: bf16 operands, fp32 accumulate            */
  BEST_PREC_FP32_TC = 2 /* the exact path's structure (fp64 chain state and algebra, one GEMM per layer) with every
                         GEMM on the tensor cores at fp32 accuracy: operands split into fp16 pairs, three MMAs per
                         product, four fp32 accumulators (north_star "bf16/fp32 variants").  log pi / gradient within
                         rel 1e-5 of the oracle like BEST_PREC_FP32; accept decisions identical to the oracle's
                         outside |log u - log alpha| < 1e-5 (FP32: 1e-6).  Hidden widths >= 64.               */
};

/* Target  log π(θ) = −½(θ−μ)ᵀΣ⁻¹(θ−μ) + s·MLP(θ) − (θ_j − θ_i²)²/(2σ²) − pen(θ)
 * (the synthetic stand-in for the paper's emulator log_prob_fn).
 * MLP (A1b): h₀=θ; h_k = act(W_k h_{k−1} + b_k), k=1..n_affine−1; out = W_last h + b_last (scalar).
 * pen (A1e, reading R6 of "smooth exponential penalty"):
 *   t_i = γ·max(0, lo_i−θ_i, θ_i−hi_i)/(hi_i−lo_i); pen = κ Σ f(t_i);
 *   f(t) = eᵗ−1−t (t ≤ 40), continued linearly with slope e⁴⁰−1 beyond.                         */
typedef struct {
  int32_t d;               /* parameter dimension, 1..32                                         */
  int32_t n_affine;        /* number of affine maps (hidden layers + 1); 0 ⇒ no MLP term         */
  const int32_t* widths;   /* host [n_affine+1] = {d, n1, …, nK, 1}                              */
  const float* W_flat;     /* host: W_1 … W_{n_affine} concatenated, W_k row-major
                              [widths[k]][widths[k−1]]                                           */
  const float* b_flat;     /* host: b_1 … b_{n_affine} concatenated                              */
  int32_t activation;      /* BEST_ACT_*                                                         */
  float mlp_scale;         /* s                                                                  */
  const double* mu;        /* host [d]; NULL ⇒ no Gaussian term                                  */
  const double* Sigma_inv; /* host [d*d] SPD precision, row-major; factored Σ⁻¹=RᵀR in fp64      */
  const double* lo;        /* host [d] box; NULL ⇒ unbounded                                     */
  const double* hi;        /* host [d]                                                           */
  float pen_kappa, pen_gamma;
  int32_t banana_i, banana_j; /* −(θ_j − θ_i²)²/(2σ²) (A1d); banana_i < 0 ⇒ off                 */
  float banana_sigma;
  const double* L;         /* host [d*d] lower-triangular whitening factor, eq (2.4) P:L78;
                              NULL ⇒ identity.  Only the lower triangle is read.                 */
  int32_t precision;       /* BEST_PREC_*                                                        */
} best_config;

/* Build a context (host work: fp64 Cholesky of Sigma_inv, packing and upload of the weights).
 * Errors: BEST_ERR_ARG, BEST_ERR_NOT_SPD, BEST_ERR_UNSUPPORTED (bf16 path: hidden widths must be
 * equal and a multiple of 64, ≤ 512 … see DESIGN.md), BEST_ERR_CUDA, BEST_ERR_ALLOC.            */
int best_create(const best_config* cfg, best_ctx** out);
void best_destroy(best_ctx* ctx);

/* log π(θ) and ∇θ log π(θ) for n points (A1a–A1e).  theta [n*d] row-major float, host|dev;
 * logp [n] and grad [n*d] (nullable ⇒ forward only) float, host|dev.  With any host pointer the
 * call copies through the device and synchronises `stream` before returning.                    */
int best_logp_grad(best_ctx* ctx, const float* theta, int64_t n, float* logp, float* grad,
                   void* stream);

/* Chain state: n_chains chains at theta0 [n_chains*d] (float, host|dev); evaluates and caches
 * log π and ∇θ log π at θ₀; step counter 0, accept counters 0.                                   */
int best_state_create(best_ctx* ctx, int64_t n_chains, const float* theta0, void* stream,
                      best_state** out);
void best_state_destroy(best_state* st);

/* Samplers.  The Philox4x32-10 stream is keyed by (seed; chain, global step, slot) (north_star;
 * reading R1), and the state's global step counter keeps increasing across calls, so one call of
 * N steps equals k calls of N/k steps bit for bit.  trace_dev (nullable, device) receives the
 * post-accept θ every `thin` steps as float [n_steps/thin][n_chains][d]; thin ≤ 0 ⇒ no trace.
 *
 * MH   (A4; reading R5): θ' = θ + ε L ξ, ξ~N(0,1); log α = log π(θ') − log π(θ).
 * MALA (A5; eq (2.3) P:L70 in whitened space; reading R4): z' = z + ε g_z + √(2ε) ξ,
 *       g_z = Lᵀ∇θ log π; Hastings ratio with q(·|z) = N(z + ε g_z, 2ε·1).
 * HMC  (A6; eq (2.1),(2.8) P:L56, L96): q~N(0,1); n_leapfrog kick-drift-kick steps of size ε in
 *       whitened space (identity mass); log α = H(z,q) − H(z',q'); one "step" = one
 *       trajectory.
 * AIES (A7; eq (2.13)-(2.15) P:L159-168): two half-ensembles [0,B/2), [B/2,B); walker i moves
 *       against a uniformly drawn partner j of the other half: θ' = θ_j + z(θ_i − θ_j),
 *       z = (u(a−1)+1)²/a, log α = (d−1) ln z + log π(θ') − log π(θ_i); no whitening.
 * All: accept iff log u < log α (NaN ⇒ reject; reading R7).
 * Errors: BEST_ERR_ARG for eps <= 0, n_leapfrog < 1, a <= 1, odd or < 2 walker count (AIES).    */
int best_step_mh(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float eps,
                 float* trace_dev, int32_t thin, void* stream);
int best_step_mala(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float eps,
                   float* trace_dev, int32_t thin, void* stream);
int best_step_hmc(best_ctx* ctx, best_state* st, int64_t n_traj, uint64_t seed, float eps,
                  int32_t n_leapfrog, float* trace_dev, int32_t thin, void* stream);
int best_step_aies(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float a,
                   float* trace_dev, int32_t thin, void* stream);

/* the Differential Evolution move of the ensemble sampler, eq (2.16):
 *   x_i' = x_i + gamma (x_j - x_k),  gamma = (1 + eta) 2.38 / sqrt(2 d),  eta ~ N(0, sigma_gamma).
 * Same ensemble split, update order, state, trace and step counter as best_step_aies (half 0 against
 * the current half 1, then half 1 against the updated half 0; one step = B forward evaluations).
 * DESIGN.md reading R23: j != k are drawn uniformly from the OTHER half (control block words 2, 3),
 * eta = sigma_gamma * (first normal of slot 1); the proposal is symmetric, so
 * log alpha = log pi(x') - log pi(x_i).  No whitening.
 * Errors: BEST_ERR_ARG for sigma_gamma < 0 (0 is allowed: fixed gamma), odd or < 4 walker count.     */
int best_step_aies_de(best_ctx* ctx, best_state* st, int64_t n_steps, uint64_t seed, float sigma_gamma,
                      float* trace_dev, int32_t thin, void* stream);

/* Running covariance adaptation (A9; reading R14).  While adapt_every > 0 the
 * MH/MALA/HMC steps of `st` accumulate n, Σθ, Σθθᵀ (fp64) of the post-accept states of all chains;
 * every adapt_every steps  C = scatter/(n−1),  C_ii *= (1+jitter),  L = chol(C)  is computed ON
 * DEVICE and replaces the context's whitening factor (jitter×10 retries up to 5 times, else L is
 * kept).  The window (sums, step count, buffers) belongs to `st`: other states of the context neither
 * feed nor disturb it.  adapt_every = 0 switches it off; every call with adapt_every > 0 opens a fresh
 * window.  Not used by AIES.  Synchronises the device.                                   */
int best_set_adaptation(best_ctx* ctx, best_state* st, int32_t adapt_every, double jitter);
/* Multi-GPU adaptation (chains are sharded over ranks with no per-step traffic; "covariance
 * adaptation = one all-reduce of d^2+d+1 fp64 values per window"; the covariance is that of the
 * whole ensemble of chains).  With an exchange function set, every window of `st` closes as
 *   own sums -> packet [ n | ref (d) | sum(theta-ref) (d) | sum (theta-ref)(theta-ref)^T (d*d) ]   (np = 1+2d+d*d
 *   doubles; each rank's sums are about its own reference point `ref`)
 *   -> fn(send_dev, recv_dev, np, stream, user): an ALL-GATHER over the job's ranks, rank r's packet to
 *      recv_dev[r*np .. r*np+np), enqueued on `stream` (e.g. ncclAllGather, or torch.distributed
 *      all_gather_into_tensor under that stream); both pointers are device memory owned by the library;
 *      return 0, anything else makes the step call fail with BEST_ERR_CUDA
 *   -> the library moves every packet to rank 0's reference point, adds them in rank order (identical bits
 *      on all ranks) and computes C, L = chol(C) as in best_set_adaptation from the sums of ALL ranks.
 * Every rank must close its windows at the same steps (same adapt_every, same step calls).  world_size >= 1;
 * fn = NULL switches the exchange off.  Allocates (1 + world_size) * np doubles, once.  The callback is called
 * on the host thread inside best_step_* / best_burn_in.  Errors: BEST_ERR_ARG, BEST_ERR_ALLOC.               */
typedef int (*best_exchange_fn)(const double* send_dev, double* recv_dev, int64_t count, void* stream, void* user);
int best_set_adaptation_exchange(best_state* st, best_exchange_fn fn, void* user, int32_t world_size);
/* Ensemble moves sharded over ranks ("AIES = one all-gather of the complementary half's positions per
 * half-step").  Every rank holds the WHOLE ensemble in `st` (same theta0, chain offset 0 on all ranks: walker i
 * draws the Philox stream of walker i whichever rank moves it).  With an exchange function set, best_step_aies
 * and best_step_aies_de move only walkers [rank*cnt, rank*cnt + cnt) of each half-ensemble, cnt = B/2/world_size,
 * with partners drawn from the whole other half, and after every half-step call
 *   fn(send_dev, recv_dev, (d+1)*cnt, stream, user)
 * -- an all-gather as in best_set_adaptation_exchange -- of the slice just moved ([d+1][cnt] doubles: theta rows, then
 * log pi), which the library writes into every rank's copy of that half.  After a step all ranks hold the same
 * theta and log pi, bit for bit those of the unsharded run; acceptance counters cover a rank's own walkers only.
 * Two all-gathers per step.  A trace pointer is refused (BEST_ERR_ARG) while the exchange is set.
 * Errors: BEST_ERR_ARG (B/2 not a multiple of world_size, rank outside 0..world_size-1), BEST_ERR_ALLOC.       */
int best_set_aies_exchange(best_state* st, best_exchange_fn fn, void* user, int32_t rank, int32_t world_size);
/* number of successful / failed whitening updates so far (synchronises) */
int best_adapt_stats(best_ctx* ctx, int64_t* n_updates, int64_t* n_failures);

/* Whitening factor L (host [d*d], row-major, lower triangle).  get synchronises the device.     */
int best_get_whitening(best_ctx* ctx, double* L_host);
int best_set_whitening(best_ctx* ctx, const double* L_host);

/* per-dimension step sizes (sec. 5.2: "a step size 10 times larger for the
 * extension parameters") and the hard-box prior option; readings R20, R21.
 *
 * best_set_step_scale: s_host [d] (host, copied; NULL = all ones), every s_i positive and finite else
 * BEST_ERR_ARG.  Coordinate i of the whitened space then moves with eps_i = eps * s_i in MH and in the
 * HMC leap-frog (drift and kick, i.e. a diagonal mass matrix diag(s)^-2); MALA, the one-step limit, uses
 * eq (2.3) with eps_i = eps * s_i^2 (drift eps_i g_i, noise sqrt(2 eps_i)).  AIES does not whiten and is
 * not affected.  The factors persist across best_set_whitening and covariance adaptation (A9), which
 * keep updating the unscaled factor that best_get_whitening returns.  Synchronises the device.
 *
 * best_set_hard_box: on != 0 replaces the smooth penalty (A1e) by log pi = -inf outside [lo, hi] (the
 * boundary belongs to the box), so such proposals are rejected (accept rule R7); gradients are those of
 * the remaining terms.  BEST_ERR_ARG if the context was created without a box.  Cached log pi of
 * existing states is not recomputed: call it before best_state_create (or best_state_set afterwards). */
int best_set_step_scale(best_ctx* ctx, const double* s_host);
int best_set_hard_box(best_ctx* ctx, int32_t on);

/* the burn-in loop of PAPER.md sec. 3.2 / 4 ("a burn-in loop where the covariance
 * matrix and the best-fit point are iteratively updated based on short chains"; sec. 4.3: iterations of
 * n_steps steps "of which the first [n_adapt] steps are used for step size adaptation and afterwards
 * discarded"); reading R22.  Host-side schedule around the step kernels and A9:
 * for each of n_iter iterations
 *   (1) n_adapt steps in blocks of `block` steps (the last block may be shorter); after block m the
 *       acceptance fraction alpha of ALL chains over the block (summed on the device) drives Nesterov
 *       dual averaging (Hoffman & Gelman 2014, Alg. 5: gamma 0.05, t0 10, kappa 0.75, mu = log(10 eps)),
 *       restarted from the current eps; the next block runs with eps_m, the iteration ends with the
 *       averaged step exp(log eps-bar), rounded to float;
 *   (2) n_steps - n_adapt steps with one covariance window over all of them; at its end the whitening
 *       factor is replaced on the device (A9, `jitter` as in best_set_adaptation);
 *   (3) the chain with the largest cached log pi updates the best-fit point if it beats the previous
 *       iterations.
 * method: BEST_METHOD_MH / _MALA / _HMC (the paper runs no burn-in loop for AIES: BEST_ERR_ARG);
 * n_leapfrog is read for HMC only.  *eps_inout (host): initial step in, adapted step out.
 * target_accept in (0,1), e.g. 0.234 MH, 0.574 MALA, 0.65-0.8 HMC.  best_theta [d] / best_logp (host,
 * nullable) receive the best-fit point in the original space (fp32 / fp64).  eps_hist (host, nullable,
 * capacity n_iter * ceil(n_adapt / block)) receives the step used in every adaptation block.
 * Synchronises `stream` after every block; leaves adaptation switched off.  The global step counter
 * advances by n_iter * n_steps.                                                                       */
/* the Gelman-Rubin type convergence statistic R - 1 of PAPER.md eq (4.1)-(4.2), on the
 * device, from a trace as written by best_step_* (`trace_dev`: device, fp32, [n][B][d]: n samples of each
 * of B chains).  B = covariance of the chain means, W = mean of the within-chain covariances (both
 * unbiased), d_i = sqrt(B_ii), R - 1 = max |eig((D^-1 W D^-1)^-1 (D^-1 B D^-1))|.  fp64 accumulation with
 * a fixed summation order (same trace => same bits).  `*rminus1_host` (host) receives the value.
 * Synchronises `stream`.  Errors: BEST_ERR_ARG for n < 2, B < 2, d outside 1..32 or a host trace pointer;
 * BEST_ERR_NOT_SPD (value NaN) if W, in units of the between-chain variance, is not positive definite to
 * 1e-12 (e.g. a dimension in which no chain ever moved: R - 1 > 1e12 is not resolvable) or some B_ii = 0. */
int best_rminus1(const float* trace_dev, int64_t n, int64_t B, int32_t d, double* rminus1_host, void* stream);

/* best_rminus1 for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same kernels, grids and summation order (hence the same bits, PAPER.md eq
 * (4.1)-(4.2)), with the scratch in a file-scope `static __device__` array of 2^20 doubles (8 MiB, held by every
 * GPU that loads the library until exit).  Calls no cudaMalloc / cudaMallocAsync / cudaFree; the first call on a
 * device looks the array's device address up (cudaGetSymbolAddress) and caches it.  Arguments as best_rminus1.
 * Limit: B*d + d + (min(ceil(n*B/64), 592) + min(ceil(B/64), 148))*d*d + 2 <= best_rminus1_noalloc_max_doubles()
 * (e.g. B <= 18 800 chains at d = 27, B <= 9 000 at d = 32, any n); larger traces return BEST_ERR_ARG with the
 * sizes in best_last_error() -- use best_rminus1.  All calls on one device SHARE the array, which keeps the last
 * call's contents (every word a call reads is first written by that call, nothing needs clearing): calls that
 * overlap on the GPU (two streams or two host threads) race.  Synchronises `stream`.  Other errors as
 * best_rminus1, BEST_ERR_CUDA if the symbol lookup fails.                                                     */
int best_rminus1_noalloc(const float* trace_dev, int64_t n, int64_t B, int32_t d, double* rminus1_host, void* stream);
int64_t best_rminus1_noalloc_max_doubles(void);

/* Measurement aid for the small-batch roofline ("measure the box's L2 bandwidth with a
 * resident-copy microbenchmark"; the small-batch path streams the weight packs from L2, sec. 3.1
 * "evaluating the emulator for up to 100 points simultaneously does not affect the evaluation time").
 * One CTA of 512 threads per SM reads a freshly allocated device buffer of `bytes` (1 MiB..96 MiB, multiple
 * of 8 KiB: resident in the 126 MB L2 after an untimed first pass) `passes` times with 16-byte loads;
 * `*gb_per_s_host` (host) receives bytes * passes * CTAs / CUDA-event time.  Allocates and frees its buffer,
 * synchronises `stream`.  Errors: BEST_ERR_ARG (sizes), BEST_ERR_CUDA.                                    */
int best_probe_l2_read(int64_t bytes, int32_t passes, double* gb_per_s_host, void* stream);

enum { BEST_METHOD_MH = 0, BEST_METHOD_MALA = 1, BEST_METHOD_HMC = 2 };
int best_burn_in(best_ctx* ctx, best_state* st, int32_t method, int32_t n_iter, int64_t n_steps,
                 int64_t n_adapt, int64_t block, uint64_t seed, float* eps_inout, float target_accept,
                 int32_t n_leapfrog, double jitter, float* best_theta, double* best_logp,
                 float* eps_hist, void* stream);

/* Read the state back (all pointers host, each nullable): theta [B*d], logp [B], grad [B*d]
 * (float, original space), global step counter, per-chain accept counters [B], total emulator
 * evaluations.  Synchronises `stream`.  After MH / ensemble steps the gradient cache is stale: asking
 * for `grad` then evaluates it (counted in n_evals) WITHOUT touching the cached log π, so a read-back
 * between two step calls never changes the chain.                                                  */
int best_state_get(best_state* st, float* theta, float* logp, float* grad, uint64_t* step,
                   uint64_t* n_accept, uint64_t* n_evals, void* stream);
/* Same state in the library's internal precision (fp64 on the fp32 path): exact checkpoints.    */
int best_state_get_f64(best_state* st, double* theta, double* logp, double* grad, void* stream);
/* log α of every chain's most recent proposal (host [B]); synchronises.  Diagnostics / tests.   */
int best_state_last_log_alpha(best_state* st, double* log_alpha, void* stream);
/* Overwrite θ (host|dev float [B*d]) and the step counter; recomputes log π and ∇θ log π;
 * accept counters are kept.                                                                     */
int best_state_set(best_state* st, const float* theta, uint64_t step, void* stream);
/* Multi-GPU sharding (chains are independent units, partitioned over ranks with no data-path
 * collective).  Chain c of `st` draws the Philox stream of GLOBAL chain id chain0 + c (counter word 0 of
 * reading R1), so rank r of a job holding B chains per rank sets chain0 = r*B and the ranks' streams are
 * disjoint, while chain0 = 0 (the default) reproduces the single-process stream.  For the ensemble moves the
 * partner indices stay local to the state (one independent ensemble per state).
 * Errors: BEST_ERR_ARG if chain0 + n_chains > 2^32.                                                       */
int best_state_set_chain_offset(best_state* st, uint64_t chain0);

/* Number of kernels this library has launched so far in this process (all contexts). */
uint64_t best_launch_count(void);
const char* best_last_error(void);
const char* best_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BEST_H_ */
