// fp32 emulator path (A1b forward, A1c input-gradient) on the FP32 FMA pipe.
// Layer-by-layer register-tiled GEMMs with fused bias/activation (forward) and act' (backward)
// epilogues; activations live in L2-resident global scratch.  This is the exact path that the
// 1e-5 parity and accept-bit tests run on; the tensor-core path is tc_fused.cu.
#include "best_internal.h"

namespace best {
namespace {

constexpr int BM = 128, BN = 64, BK = 16, NT = 256;

enum { EPI_FWD_ACT = 0, EPI_BWD_MUL = 1, EPI_PLAIN = 2 };

__device__ __forceinline__ void act_eval(int kind, float a, float& h, float& dh) {
  if (kind == BEST_ACT_TANH) {
    h = tanhf(a);
    dh = 1.0f - h * h;
  } else {  // SiLU, sigma evaluated overflow-safe
    const float e = expf(-fabsf(a));
    const float sg = (a >= 0.0f) ? 1.0f / (1.0f + e) : e / (1.0f + e);
    h = a * sg;
    dh = sg * (1.0f + a * (1.0f - sg));
  }
}

// C[M][ldc] = epi( A[M][K] * B ),  A row-major (lda).  B_NT: B given as Wt[N][K] (ldb) so that
// C = A Wt^T (forward);  !B_NT: B given as W[K][N] (ldb) so that C = A W (backward).
// All of K, N, lda, ldb, ldc are multiples of 4 (zero padded), pointers 16-byte aligned.
template <bool B_NT, int EPI>
__global__ void __launch_bounds__(NT)
sgemm_fused(const float* __restrict__ A, int lda, const float* __restrict__ Bm, int ldb,
            float* __restrict__ C, int ldc, int M, int N, int K,
            const float* __restrict__ bias,   // FWD: [N]
            float* __restrict__ aux, int ldaux,  // FWD: act' out [M][ldaux]; BWD: act' in
            int act_kind) {
  __shared__ __align__(16) float As[BK][BM + 4];
  __shared__ __align__(16) float Bs[BK][BN + 4];
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;  // tx: 4 columns each, ty: 8 rows each
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;

  float acc[8][4];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j] = 0.0f;

  for (int k0 = 0; k0 < K; k0 += BK) {
    // A tile: 128 rows x 4 float4 (along K) = 512 float4, 2 per thread
#pragma unroll
    for (int it = 0; it < 2; ++it) {
      const int idx = tid + it * NT;
      const int r = idx >> 2, c4 = (idx & 3) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (m0 + r < M && k0 + c4 < K)
        v = *reinterpret_cast<const float4*>(A + (size_t)(m0 + r) * lda + k0 + c4);
      As[c4 + 0][r] = v.x; As[c4 + 1][r] = v.y; As[c4 + 2][r] = v.z; As[c4 + 3][r] = v.w;
    }
    if (B_NT) {  // Wt[N][K]: 64 rows x 4 float4
      const int r = tid >> 2, c4 = (tid & 3) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (n0 + r < N && k0 + c4 < K)
        v = *reinterpret_cast<const float4*>(Bm + (size_t)(n0 + r) * ldb + k0 + c4);
      Bs[c4 + 0][r] = v.x; Bs[c4 + 1][r] = v.y; Bs[c4 + 2][r] = v.z; Bs[c4 + 3][r] = v.w;
    } else {     // W[K][N]: 16 rows x 16 float4
      const int r = tid >> 4, c4 = (tid & 15) * 4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (k0 + r < K && n0 + c4 < N)
        v = *reinterpret_cast<const float4*>(Bm + (size_t)(k0 + r) * ldb + n0 + c4);
      *reinterpret_cast<float4*>(&Bs[r][c4]) = v;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      const float4 a0 = *reinterpret_cast<const float4*>(&As[k][ty * 8]);
      const float4 a1 = *reinterpret_cast<const float4*>(&As[k][ty * 8 + 4]);
      const float4 b0 = *reinterpret_cast<const float4*>(&Bs[k][tx * 4]);
      const float a[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
      const float b[4] = {b0.x, b0.y, b0.z, b0.w};
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }

  const int n = n0 + tx * 4;
  if (n >= N) return;
  float4 bv = make_float4(0.f, 0.f, 0.f, 0.f);
  if (EPI == EPI_FWD_ACT) bv = *reinterpret_cast<const float4*>(bias + n);
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int m = m0 + ty * 8 + i;
    if (m >= M) continue;
    float4 o;
    if (EPI == EPI_FWD_ACT) {
      float4 dv;
      act_eval(act_kind, acc[i][0] + bv.x, o.x, dv.x);
      act_eval(act_kind, acc[i][1] + bv.y, o.y, dv.y);
      act_eval(act_kind, acc[i][2] + bv.z, o.z, dv.z);
      act_eval(act_kind, acc[i][3] + bv.w, o.w, dv.w);
      *reinterpret_cast<float4*>(aux + (size_t)m * ldaux + n) = dv;
    } else if (EPI == EPI_BWD_MUL) {
      const float4 dv = *reinterpret_cast<const float4*>(aux + (size_t)m * ldaux + n);
      o = make_float4(acc[i][0] * dv.x, acc[i][1] * dv.y, acc[i][2] * dv.z, acc[i][3] * dv.w);
    } else {
      o = make_float4(acc[i][0], acc[i][1], acc[i][2], acc[i][3]);
    }
    *reinterpret_cast<float4*>(C + (size_t)m * ldc + n) = o;
  }
}

// Output layer (N = 1): out[m] = w . H[m] + b; and the first backward operand
// delta[m][n] = w[n] * act'[m][n].  One warp per row.
__global__ void out_and_delta(const float* __restrict__ H, const float* __restrict__ Dact, int ld,
                              int K, const float* __restrict__ w, const float* __restrict__ b,
                              float* __restrict__ out, float* __restrict__ delta, int M,
                              int want_grad) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= M) return;
  const float* h = H + (size_t)warp * ld;
  float s = 0.0f;
  for (int k = lane; k < K; k += 32) s = fmaf(h[k], w[k], s);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) out[warp] = s + b[0];
  if (want_grad) {
    const float* dd = Dact + (size_t)warp * ld;
    float* de = delta + (size_t)warp * ld;
    for (int k = lane; k < K; k += 32) de[k] = w[k] * dd[k];
  }
}

// MLP with no hidden layer (n_affine == 1): out = W1 x + b, grad = W1.
__global__ void affine_only(const float* __restrict__ X, int ld, int K, const float* __restrict__ w,
                            const float* __restrict__ b, float* __restrict__ out,
                            float* __restrict__ grad, int M, int want_grad) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= M) return;
  float s = b[0];
  for (int k = 0; k < K; ++k) s = fmaf(X[(size_t)m * ld + k], w[k], s);
  out[m] = s;
  if (want_grad)
    for (int k = 0; k < K; ++k) grad[(size_t)m * ld + k] = w[k];
}

template <bool B_NT, int EPI>
void launch_gemm(const float* A, int lda, const float* Bm, int ldb, float* C, int ldc, int M, int N,
                 int K, const float* bias, float* aux, int ldaux, int act, cudaStream_t s) {
  dim3 grid((N + BN - 1) / BN, (M + BM - 1) / BM);
  sgemm_fused<B_NT, EPI><<<grid, NT, 0, s>>>(A, lda, Bm, ldb, C, ldc, M, N, K, bias, aux, ldaux, act);
  count_launch();
}

}  // namespace

int mlp_fp32_reserve(best_ctx* ctx, int64_t n) {
  if (ctx->n_affine == 0 || n <= ctx->scratch_n) return BEST_OK;
  auto freep = [](float*& p) { if (p) cudaFree(p); p = nullptr; };
  freep(ctx->X0); freep(ctx->delta[0]); freep(ctx->delta[1]); freep(ctx->mlp_out); freep(ctx->mlp_grad);
  for (auto& p : ctx->H) freep(p);
  for (auto& p : ctx->Dact) freep(p);
  ctx->scratch_n = 0;
  const int nh = ctx->n_affine - 1;
  ctx->H.assign(nh, nullptr);
  ctx->Dact.assign(nh, nullptr);
  int maxw = ctx->dp;
  for (int k = 1; k <= nh; ++k) maxw = ctx->wp[k] > maxw ? ctx->wp[k] : maxw;
  BEST_CUDA(cudaMalloc(&ctx->X0, sizeof(float) * n * ctx->dp));
  BEST_CUDA(cudaMalloc(&ctx->mlp_out, sizeof(float) * n));
  BEST_CUDA(cudaMalloc(&ctx->mlp_grad, sizeof(float) * n * ctx->dp));
  const int64_t nl = n;
  for (int k = 0; k < nh; ++k) {
    BEST_CUDA(cudaMalloc(&ctx->H[k], sizeof(float) * nl * ctx->wp[k + 1]));
    BEST_CUDA(cudaMalloc(&ctx->Dact[k], sizeof(float) * nl * ctx->wp[k + 1]));
  }
  BEST_CUDA(cudaMalloc(&ctx->delta[0], sizeof(float) * nl * maxw));
  BEST_CUDA(cudaMalloc(&ctx->delta[1], sizeof(float) * nl * maxw));
  ctx->scratch_n = n;
  return BEST_OK;
}

// forward (+ input gradient) of M points: X [M][dp] -> out [M], grad [M][dp]; layer buffers hold >= M rows
static int run_chain(best_ctx* ctx, int M, const float* X, float* out, float* grad, bool want_grad, cudaStream_t s) {
  const int nh = ctx->n_affine - 1;  // hidden layers
  const float* in = X;
  int ldin = ctx->dp;
  for (int k = 0; k < nh; ++k) {  // h_k = act(W_k h_{k-1} + b_k)
    if (ctx->tc32)
      BEST_TRY(tc32_gemm(ctx, true, k, in, ldin, ctx->H[k], ctx->wp[k + 1], M, ctx->b[k], ctx->Dact[k],
                         ctx->wp[k + 1], EPI_FWD_ACT, s));
    else
      launch_gemm<true, EPI_FWD_ACT>(in, ldin, ctx->W[k], ctx->wp[k], ctx->H[k], ctx->wp[k + 1], M,
                                     ctx->wp[k + 1], ctx->wp[k], ctx->b[k], ctx->Dact[k],
                                     ctx->wp[k + 1], ctx->activation, s);
    in = ctx->H[k];
    ldin = ctx->wp[k + 1];
  }
  {
    const int threads = 256, rows_per_block = threads / 32;
    out_and_delta<<<(M + rows_per_block - 1) / rows_per_block, threads, 0, s>>>(
        ctx->H[nh - 1], ctx->Dact[nh - 1], ctx->wp[nh], ctx->wp[nh], ctx->W[nh], ctx->b[nh],
        out, ctx->delta[0], M, want_grad ? 1 : 0);
    count_launch();
  }
  if (want_grad) {
    int cur = 0;
    for (int k = nh - 1; k >= 1; --k) {  // delta_k = (delta_{k+1} W_{k+1}) .* act'(a_k)
      if (ctx->tc32)
        BEST_TRY(tc32_gemm(ctx, false, k, ctx->delta[cur], ctx->wp[k + 1], ctx->delta[cur ^ 1], ctx->wp[k], M,
                           nullptr, ctx->Dact[k - 1], ctx->wp[k], EPI_BWD_MUL, s));
      else
        launch_gemm<false, EPI_BWD_MUL>(ctx->delta[cur], ctx->wp[k + 1], ctx->W[k], ctx->wp[k],
                                        ctx->delta[cur ^ 1], ctx->wp[k], M, ctx->wp[k], ctx->wp[k + 1],
                                        nullptr, ctx->Dact[k - 1], ctx->wp[k], ctx->activation, s);
      cur ^= 1;
    }
    if (ctx->tc32)
      BEST_TRY(tc32_gemm(ctx, false, 0, ctx->delta[cur], ctx->wp[1], grad, ctx->dp, M, nullptr, nullptr, 0,
                         EPI_PLAIN, s));
    else
      launch_gemm<false, EPI_PLAIN>(ctx->delta[cur], ctx->wp[1], ctx->W[0], ctx->wp[0], grad,
                                    ctx->dp, M, ctx->dp, ctx->wp[1], nullptr, nullptr, 0, 0, s);
  }
  return BEST_OK;
}

int mlp_fp32_run(best_ctx* ctx, int64_t n, bool want_grad, cudaStream_t s) {
  const int nh = ctx->n_affine - 1;  // hidden layers
  const int M = (int)n;
  if (nh == 0) {
    affine_only<<<(M + 127) / 128, 128, 0, s>>>(ctx->X0, ctx->dp, ctx->d, ctx->W[0], ctx->b[0],
                                                ctx->mlp_out, ctx->mlp_grad, M, want_grad ? 1 : 0);
    count_launch();
    BEST_CUDA(cudaGetLastError());
    return BEST_OK;
  }
  // (Row chunks that keep the fp32 layer buffers L2-resident were measured on the tensor-core variant: each GEMM's
  // epilogue drops from 20-24 k to 9 k cycles per CTA, but four times the launches cost more than that saves.)
  BEST_TRY(run_chain(ctx, M, ctx->X0, ctx->mlp_out, ctx->mlp_grad, want_grad, s));
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

}  // namespace best
