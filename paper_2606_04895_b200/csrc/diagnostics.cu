// the Gelman-Rubin type statistic R - 1 of PAPER.md eq (4.1)-(4.2) on the device, from a
// trace [n][B][d] (fp32, as written by best_step_*).  With m_c the chain means, m their mean and
//   S = sum_{t,c} (x_tc - m)(x_tc - m)^T,   M = sum_c (m_c - m)(m_c - m)^T :
//   B = M / (B - 1)  (covariance of the chain means),   W = (S - n M) / (B (n - 1))  (mean chain covariance),
//   d_i = sqrt(B_ii),  B~ = D^-1 B D^-1,  W~ = D^-1 W D^-1,  R - 1 = max |eig(W~^-1 B~)|.
// W~ = L L^T is SPD and B~ symmetric, so the eigenvalues are those of the symmetric L^-1 B~ L^-T (cyclic
// Jacobi).  Everything is accumulated in fp64; partial sums are combined in a fixed order.
#include <algorithm>

#include "best_internal.h"

namespace best {
namespace {

constexpr int G_TPB = 128;

// means[c*d + i] = (1/n) sum_t trace[t][c][i]   (one thread per (c, i): fully coalesced over the trace row)
__global__ void k_chain_means(const float* __restrict__ trace, int64_t n, int64_t row, double* __restrict__ means) {
  const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= row) return;
  double s = 0.0;
  for (int64_t t = 0; t < n; ++t) s += (double)trace[t * row + e];
  means[e] = s / (double)n;
}

// gm[i] = (1/B) sum_c means[c][i]   (one block; thread i sums its dimension in chain order)
__global__ void k_grand_mean(const double* __restrict__ means, int64_t B, int d, double* __restrict__ gm) {
  const int i = threadIdx.x;
  if (i >= d) return;
  double s = 0.0;
  for (int64_t c = 0; c < B; ++c) s += means[c * d + i];
  gm[i] = s / (double)B;
}

// acc[blk][i*d + j] = sum over the block's rows of (x_i - ref_i)(x_j - ref_j); rows are [nrows][d]
template <typename T>
__global__ void __launch_bounds__(G_TPB)
k_gram_partial(const T* __restrict__ rows, int64_t nrows, int d, const double* __restrict__ ref,
               double* __restrict__ acc) {
  extern __shared__ double xs[];  // [G_TPB][d + 1]
  const int dd = d * d, pitch = d + 1;
  double mine[(kMaxD * kMaxD + G_TPB - 1) / G_TPB];
#pragma unroll
  for (int q = 0; q < (kMaxD * kMaxD + G_TPB - 1) / G_TPB; ++q) mine[q] = 0.0;
  for (int64_t r0 = blockIdx.x * (int64_t)G_TPB; r0 < nrows; r0 += (int64_t)gridDim.x * G_TPB) {
    const int nv = (int)((nrows - r0 < G_TPB) ? (nrows - r0) : G_TPB);
    __syncthreads();
    for (int e = threadIdx.x; e < nv * d; e += G_TPB) {   // contiguous, coalesced
      const int r = e / d, i = e - r * d;
      xs[r * pitch + i] = (double)rows[r0 * d + e] - ref[i];
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < (kMaxD * kMaxD + G_TPB - 1) / G_TPB; ++q) {
      const int e = threadIdx.x + q * G_TPB;
      if (e < dd) {
        const int i = e / d, j = e - i * d;
        double s = 0.0;
        for (int r = 0; r < nv; ++r) s += xs[r * pitch + i] * xs[r * pitch + j];
        mine[q] += s;
      }
    }
  }
#pragma unroll
  for (int q = 0; q < (kMaxD * kMaxD + G_TPB - 1) / G_TPB; ++q) {
    const int e = threadIdx.x + q * G_TPB;
    if (e < dd) acc[(size_t)blockIdx.x * dd + e] = mine[q];
  }
}

// out[0] = R - 1, out[1] = status (0 ok, 1 W~ not positive definite / B_ii = 0)
__global__ void k_rminus1_finalize(const double* __restrict__ accS, int nblkS, const double* __restrict__ accM,
                                   int nblkM, int d, double n, double nb, double* __restrict__ out) {
  __shared__ double S[kMaxD * kMaxD], M[kMaxD * kMaxD], A[kMaxD * kMaxD], Lc[kMaxD * kMaxD];
  const int dd = d * d;
  for (int e = threadIdx.x; e < dd; e += blockDim.x) {
    double s = 0.0, m = 0.0;
    for (int b = 0; b < nblkS; ++b) s += accS[(size_t)b * dd + e];
    for (int b = 0; b < nblkM; ++b) m += accM[(size_t)b * dd + e];
    S[e] = s; M[e] = m;
  }
  __syncthreads();
  if (threadIdx.x != 0) return;
  bool ok = true;
  // W~ into S, B~ into M (symmetrised)
  for (int i = 0; i < d; ++i)
    for (int j = 0; j <= i; ++j) {
      const double mij = 0.5 * (M[i * d + j] + M[j * d + i]), sij = 0.5 * (S[i * d + j] + S[j * d + i]);
      const double bij = mij / (nb - 1.0), wij = (sij - n * mij) / (nb * (n - 1.0));
      A[i * d + j] = A[j * d + i] = bij;
      Lc[i * d + j] = Lc[j * d + i] = wij;
    }
  for (int i = 0; i < d; ++i) if (!(A[i * d + i] > 0.0)) ok = false;
  if (ok) {
    for (int i = 0; i < d; ++i)
      for (int j = 0; j < d; ++j) {
        const double sc = sqrt(A[i * d + i]) * sqrt(A[j * d + j]);
        M[i * d + j] = A[i * d + j] / sc;
        S[i * d + j] = Lc[i * d + j] / sc;
      }
    // Cholesky W~ = L L^T (lower, in Lc)
    for (int j = 0; j < d && ok; ++j) {
      double s = S[j * d + j];
      for (int k = 0; k < j; ++k) s -= Lc[j * d + k] * Lc[j * d + k];
      // W~ is in units of the between-chain variance: a pivot below 1e-12 means R - 1 > 1e12, which the
      // fp64 cancellation S - n M cannot resolve (a dimension in which no chain moved), or a singular W
      if (!(s > 1e-12) || !(s > 1e-13 * S[j * d + j])) { ok = false; break; }
      const double ljj = sqrt(s);
      Lc[j * d + j] = ljj;
      for (int i = j + 1; i < d; ++i) {
        double t = S[i * d + j];
        for (int k = 0; k < j; ++k) t -= Lc[i * d + k] * Lc[j * d + k];
        Lc[i * d + j] = t / ljj;
      }
    }
  }
  if (!ok) { out[0] = nan(""); out[1] = 1.0; return; }
  // A = L^-1 B~ L^-T : first Y = L^-1 B~ (columns), then A = Y L^-T  <=>  A^T = L^-1 Y^T
  for (int c = 0; c < d; ++c)
    for (int i = 0; i < d; ++i) {
      double t = M[i * d + c];
      for (int k = 0; k < i; ++k) t -= Lc[i * d + k] * A[k * d + c];
      A[i * d + c] = t / Lc[i * d + i];
    }
  for (int r = 0; r < d; ++r)      // row r of Y: solve L z = Y[r][:]^T, store as row r of the result
    for (int i = 0; i < d; ++i) {
      double t = A[r * d + i];
      for (int k = 0; k < i; ++k) t -= Lc[i * d + k] * S[r * d + k];
      S[r * d + i] = t / Lc[i * d + i];
    }
  for (int i = 0; i < d; ++i)
    for (int j = 0; j <= i; ++j) A[i * d + j] = A[j * d + i] = 0.5 * (S[i * d + j] + S[j * d + i]);
  // cyclic Jacobi on the symmetric A
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int i = 0; i < d; ++i) {
      diag += A[i * d + i] * A[i * d + i];
      for (int j = 0; j < i; ++j) off += A[i * d + j] * A[i * d + j];
    }
    if (off <= 1e-30 * diag || off == 0.0) break;
    for (int p = 0; p < d - 1; ++p)
      for (int q = p + 1; q < d; ++q) {
        const double apq = A[p * d + q];
        if (apq == 0.0) continue;
        const double theta = (A[q * d + q] - A[p * d + p]) / (2.0 * apq);
        const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
        const double cs = 1.0 / sqrt(t * t + 1.0), sn = t * cs;
        for (int k = 0; k < d; ++k) {   // columns p, q
          const double akp = A[k * d + p], akq = A[k * d + q];
          A[k * d + p] = cs * akp - sn * akq;
          A[k * d + q] = sn * akp + cs * akq;
        }
        for (int k = 0; k < d; ++k) {   // rows p, q
          const double apk = A[p * d + k], aqk = A[q * d + k];
          A[p * d + k] = cs * apk - sn * aqk;
          A[q * d + k] = sn * apk + cs * aqk;
        }
      }
  }
  double best = 0.0;
  for (int i = 0; i < d; ++i) best = fmax(best, fabs(A[i * d + i]));
  out[0] = best;
  out[1] = 0.0;
}

}  // namespace
}  // namespace best

using namespace best;

extern "C" int best_rminus1(const float* trace_dev, int64_t n, int64_t B, int32_t d, double* rminus1_host,
                            void* stream) {
  if (!trace_dev || !rminus1_host || n < 2 || B < 2 || d < 1 || d > kMaxD) {
    set_error("best_rminus1: need a trace with n >= 2 samples, B >= 2 chains, 1 <= d <= 32");
    return BEST_ERR_ARG;
  }
  if (!is_device_ptr(trace_dev)) { set_error("best_rminus1: trace must be a device pointer"); return BEST_ERR_ARG; }
  cudaStream_t s = (cudaStream_t)stream;
  const int dd = d * d;
  const int64_t row = B * (int64_t)d;
  const int nblkS = (int)std::min<int64_t>((n * B + G_TPB - 1) / G_TPB, 1184);
  const int nblkM = (int)std::min<int64_t>((B + G_TPB - 1) / G_TPB, 148);
  double* buf = nullptr;
  const size_t n_means = (size_t)row, n_tot = n_means + (size_t)d + (size_t)(nblkS + nblkM) * dd + 2;
  BEST_TRY(dev_alloc(&buf, n_tot));
  double *means = buf, *gm = means + n_means, *accS = gm + d, *accM = accS + (size_t)nblkS * dd,
         *out = accM + (size_t)nblkM * dd;
  auto done = [&](int rc) { cudaFree(buf); return rc; };
  k_chain_means<<<(unsigned)((row + 255) / 256), 256, 0, s>>>(trace_dev, n, row, means);
  k_grand_mean<<<1, 32, 0, s>>>(means, B, d, gm);
  const size_t smem = sizeof(double) * G_TPB * (d + 1);
  k_gram_partial<float><<<nblkS, G_TPB, smem, s>>>(trace_dev, n * B, d, gm, accS);
  k_gram_partial<double><<<nblkM, G_TPB, smem, s>>>(means, B, d, gm, accM);
  k_rminus1_finalize<<<1, 256, 0, s>>>(accS, nblkS, accM, nblkM, d, (double)n, (double)B, out);
  count_launch(5);
  double h[2] = {0.0, 0.0};
  if (cudaGetLastError() != cudaSuccess || cudaMemcpyAsync(h, out, sizeof(h), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaStreamSynchronize(s) != cudaSuccess) {
    set_error("best_rminus1: CUDA failure");
    cudaGetLastError();
    return done(BEST_ERR_CUDA);
  }
  *rminus1_host = h[0];
  if (h[1] != 0.0) {
    set_error("best_rminus1: the mean chain covariance is not positive definite (or some chain means coincide)");
    return done(BEST_ERR_NOT_SPD);
  }
  return done(BEST_OK);
}
