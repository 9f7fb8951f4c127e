// the Gelman-Rubin type statistic R - 1 of PAPER.md eq (4.1)-(4.2) on the device, from a
// trace [n][B][d] (fp32, as written by best_step_*).  With m_c the chain means, m their mean and
//   S = sum_{t,c} (x_tc - m)(x_tc - m)^T,   M = sum_c (m_c - m)(m_c - m)^T :
//   B = M / (B - 1)  (covariance of the chain means),   W = (S - n M) / (B (n - 1))  (mean chain covariance),
//   d_i = sqrt(B_ii),  B~ = D^-1 B D^-1,  W~ = D^-1 W D^-1,  R - 1 = max |eig(W~^-1 B~)|.
// W~ = L L^T is SPD and B~ symmetric, so the eigenvalues are those of the symmetric L^-1 B~ L^-T (cyclic
// Jacobi).  Everything is accumulated in fp64; partial sums are combined in a fixed order.
#include <algorithm>
#include <mutex>

#include "best_internal.h"
#include "gram.cuh"

namespace best {
namespace {

// means[c*d + i] = (1/n) sum_t trace[t][c][i]   (one thread per (c, i): fully coalesced over the trace row)
__global__ void k_chain_means(const float* __restrict__ trace, int64_t n, int64_t row, double* __restrict__ means) {
  const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= row) return;
  double s = 0.0;
  for (int64_t t = 0; t < n; ++t) s += (double)trace[t * row + e];
  means[e] = s / (double)n;
}

// gm[i] = (1/B) sum_c means[c][i]   (one block of 32 x 32 threads: part p sums the chains c = p mod 32 in
// order, the 32 parts are then added in order -- a fixed summation order)
__global__ void k_grand_mean(const double* __restrict__ means, int64_t B, int d, double* __restrict__ gm) {
  __shared__ double part[32][33];
  const int i = threadIdx.x & 31, p = threadIdx.x >> 5;
  double s = 0.0;
  if (i < d)
    for (int64_t c = p; c < B; c += 32) s += means[c * d + i];
  part[p][i] = s;
  __syncthreads();
  if (p == 0 && i < d) {
    double t = 0.0;
    for (int q = 0; q < 32; ++q) t += part[q][i];
    gm[i] = t / (double)B;
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
  if (threadIdx.x >= 32) return;          // one warp does the dense d x d algebra (lane = row / column)
  const int lane = threadIdx.x;
  __shared__ int ok_s;
  if (lane == 0) {
    bool ok = true;
    // B into A, W into Lc (symmetrised)
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
          M[i * d + j] = A[i * d + j] / sc;   // B~
          S[i * d + j] = Lc[i * d + j] / sc;  // W~
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
    ok_s = ok ? 1 : 0;
  }
  __syncwarp();
  if (!ok_s) {
    if (lane == 0) { out[0] = nan(""); out[1] = 1.0; }
    return;
  }
  // A = L^-1 B~ L^-T : Y = L^-1 B~ (lane = column), then row r of the result solves L z = Y[r][:]^T (lane = row)
  if (lane < d) {
    const int c = lane;
    for (int i = 0; i < d; ++i) {
      double t = M[i * d + c];
      for (int k = 0; k < i; ++k) t -= Lc[i * d + k] * A[k * d + c];
      A[i * d + c] = t / Lc[i * d + i];
    }
  }
  __syncwarp();
  if (lane < d) {
    const int r = lane;
    for (int i = 0; i < d; ++i) {
      double t = A[r * d + i];
      for (int k = 0; k < i; ++k) t -= Lc[i * d + k] * S[r * d + k];
      S[r * d + i] = t / Lc[i * d + i];
    }
  }
  __syncwarp();
  if (lane < d)
    for (int j = 0; j < d; ++j) A[lane * d + j] = 0.5 * (S[lane * d + j] + S[j * d + lane]);
  __syncwarp();
  // cyclic Jacobi on the symmetric A; every lane computes the same rotation, lane k updates row / column k
  for (int sweep = 0; sweep < 60; ++sweep) {
    double off = 0.0, diag = 0.0;
    for (int i = 0; i < d; ++i) {       // same fixed-order sums on every lane
      diag += A[i * d + i] * A[i * d + i];
      for (int j = 0; j < i; ++j) off += A[i * d + j] * A[i * d + j];
    }
    if (off <= 1e-30 * diag || off == 0.0) break;
    for (int p = 0; p < d - 1; ++p)
      for (int q = p + 1; q < d; ++q) {
        const double apq = A[p * d + q], app = A[p * d + p], aqq = A[q * d + q];
        __syncwarp();
        if (apq == 0.0) continue;
        const double theta = (aqq - app) / (2.0 * apq);
        const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
        const double cs = 1.0 / sqrt(t * t + 1.0), sn = t * cs;
        if (lane < d) {   // columns p, q of row `lane`
          const double akp = A[lane * d + p], akq = A[lane * d + q];
          A[lane * d + p] = cs * akp - sn * akq;
          A[lane * d + q] = sn * akp + cs * akq;
        }
        __syncwarp();
        if (lane < d) {   // rows p, q of column `lane`
          const double apk = A[p * d + lane], aqk = A[q * d + lane];
          A[p * d + lane] = cs * apk - sn * aqk;
          A[q * d + lane] = sn * apk + cs * aqk;
        }
        __syncwarp();
      }
  }
  if (lane == 0) {
    double best = 0.0;
    for (int i = 0; i < d; ++i) best = fmax(best, fabs(A[i * d + i]));
    out[0] = best;
    out[1] = 0.0;
  }
}

}  // namespace
}  // namespace best

namespace best {
namespace {
// L2 read-bandwidth probe: every CTA sweeps the WHOLE buffer `passes` times with 16-byte loads, each CTA
// starting at its own offset so that the CTAs do not walk in lockstep.  After the first touch the buffer is
// served from L2 (callers keep it well below the 126 MB).  The xor keeps the loads alive.
__global__ void __launch_bounds__(512) k_l2_read_probe(const uint4* __restrict__ buf, int64_t n16, int passes,
                                                       unsigned* __restrict__ sink) {
  unsigned acc = 0;
  const int64_t start = ((int64_t)blockIdx.x * 7919 * 512) % n16;
  for (int p = 0; p < passes; ++p) {
    for (int64_t i0 = 0; i0 < n16; i0 += 512 * 4) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        int64_t i = start + i0 + (int64_t)u * 512 + threadIdx.x;
        if (i >= n16) i -= n16;
        if (i < n16) {
          const uint4 v = __ldcg(buf + i);
          acc ^= v.x ^ v.y ^ v.z ^ v.w;
        }
      }
    }
  }
  if (acc == 0x9E3779B9u) sink[0] = acc;   // practically never; defeats dead-code elimination
}
}  // namespace
}  // namespace best

using namespace best;

extern "C" int best_probe_l2_read(int64_t bytes, int32_t passes, double* gb_per_s_host, void* stream) {
  if (!gb_per_s_host || bytes < (1 << 20) || bytes > (96ll << 20) || (bytes & 8191) || passes < 1 || passes > 1000) {
    set_error("best_probe_l2_read: 1 MiB <= bytes <= 96 MiB (multiple of 8 KiB), 1 <= passes <= 1000");
    return BEST_ERR_ARG;
  }
  cudaStream_t s = (cudaStream_t)stream;
  int dev = 0, n_sm = 0;
  BEST_CUDA(cudaGetDevice(&dev));
  BEST_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  unsigned char* buf = nullptr;
  BEST_TRY(dev_alloc(&buf, (size_t)bytes + 16));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  auto done = [&](int rc) { cudaFree(buf); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); return rc; };
  unsigned* sink = reinterpret_cast<unsigned*>(buf + bytes);
  float ms = 0.0f;
  if (cudaMemsetAsync(buf, 1, (size_t)bytes + 16, s) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
      cudaEventCreate(&e1) != cudaSuccess) { set_error("best_probe_l2_read: CUDA failure"); return done(BEST_ERR_CUDA); }
  const int64_t n16 = bytes / 16;
  k_l2_read_probe<<<n_sm, 512, 0, s>>>(reinterpret_cast<const uint4*>(buf), n16, 1, sink);   // first touch
  cudaEventRecord(e0, s);
  k_l2_read_probe<<<n_sm, 512, 0, s>>>(reinterpret_cast<const uint4*>(buf), n16, passes, sink);
  cudaEventRecord(e1, s);
  count_launch(2);
  if (cudaGetLastError() != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess ||
      cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) {
    set_error("best_probe_l2_read: CUDA failure");
    cudaGetLastError();
    return done(BEST_ERR_CUDA);
  }
  *gb_per_s_host = (double)bytes * (double)passes * (double)n_sm / ((double)ms * 1e-3) / 1e9;
  return done(BEST_OK);
}

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
  const int nblkS = (int)std::min<int64_t>((n * B + G_ROWS - 1) / G_ROWS, 592);   // 4 CTAs per SM
  const int nblkM = (int)std::min<int64_t>((B + G_ROWS - 1) / G_ROWS, 148);
  double* buf = nullptr;
  const size_t n_means = (size_t)row, n_tot = n_means + (size_t)d + (size_t)(nblkS + nblkM) * dd + 2;
  // stream-ordered allocation: cudaMalloc / cudaFree per call synchronise the device (measured: 2.7 ms calls with
  // 50-100 ms outliers)
  if (cudaMallocAsync((void**)&buf, sizeof(double) * n_tot, s) != cudaSuccess) {
    cudaGetLastError();
    set_error("best_rminus1: allocation failed");
    return BEST_ERR_ALLOC;
  }
  double *means = buf, *gm = means + n_means, *accS = gm + d, *accM = accS + (size_t)nblkS * dd,
         *out = accM + (size_t)nblkM * dd;
  auto done = [&](int rc) { cudaFreeAsync(buf, s); return rc; };
  k_chain_means<<<(unsigned)((row + 255) / 256), 256, 0, s>>>(trace_dev, n, row, means);
  k_grand_mean<<<1, 1024, 0, s>>>(means, B, d, gm);
  k_gram_partial<float><<<nblkS, G_TPB, 0, s>>>(trace_dev, n * B, d, gm, accS);
  k_gram_partial<double><<<nblkM, G_TPB, 0, s>>>(means, B, d, gm, accM);
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

// ---- best_rminus1_noalloc: the same five launches with the scratch in a file-scope device array ------------
// For callers that must not allocate (CUDA graph capture around them, serving loops, harnesses that forbid
// cudaMalloc).  Every GPU that loads the library holds these 8 MiB until exit.  All calls on a device share the
// array and it keeps the last call's contents: every word a call reads (chain means, grand mean, the Gram
// partials of the blocks it launches, the two result words) is written by that call's own kernels first, so
// nothing needs clearing -- but two calls that overlap on the GPU (two streams, two host threads) race on it.
namespace best {
namespace {
constexpr size_t kNoAllocDoubles = (size_t)1 << 20;                       // 8 MiB
static __device__ __align__(256) double g_rminus1_scratch[kNoAllocDoubles];

// In host code `g_rminus1_scratch` is only the host-side shadow of the symbol, not a device address: the device
// address is looked up once per device, with that device current, and cached.
int noalloc_scratch(double** p) {
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static double* cached[kMaxDev] = {};
  int dev = -1;
  BEST_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) { set_error("best_rminus1_noalloc: device ordinal above 63"); return BEST_ERR_ARG; }
  std::lock_guard<std::mutex> lk(mu);
  if (!cached[dev]) {
    void* sym = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&sym, g_rminus1_scratch);
    if (e != cudaSuccess || !sym) {
      cudaGetLastError();
      set_error(std::string("best_rminus1_noalloc: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e));
      return BEST_ERR_CUDA;
    }
    cached[dev] = static_cast<double*>(sym);
  }
  *p = cached[dev];
  return BEST_OK;
}
}  // namespace
}  // namespace best

extern "C" int64_t best_rminus1_noalloc_max_doubles(void) { return (int64_t)best::kNoAllocDoubles; }

extern "C" int best_rminus1_noalloc(const float* trace_dev, int64_t n, int64_t B, int32_t d, double* rminus1_host,
                                    void* stream) {
  if (!trace_dev || !rminus1_host || n < 2 || B < 2 || d < 1 || d > kMaxD) {
    set_error("best_rminus1_noalloc: need a trace with n >= 2 samples, B >= 2 chains, 1 <= d <= 32");
    return BEST_ERR_ARG;
  }
  if (!is_device_ptr(trace_dev)) {
    set_error("best_rminus1_noalloc: trace must be a device pointer");
    return BEST_ERR_ARG;
  }
  cudaStream_t s = (cudaStream_t)stream;
  const int dd = d * d;
  const int64_t row = B * (int64_t)d;
  // the same grids as best_rminus1, hence the same summation order and the same bits
  const int nblkS = (int)std::min<int64_t>((n * B + G_ROWS - 1) / G_ROWS, 592);
  const int nblkM = (int)std::min<int64_t>((B + G_ROWS - 1) / G_ROWS, 148);
  const size_t n_means = (size_t)row, n_tot = n_means + (size_t)d + (size_t)(nblkS + nblkM) * dd + 2;
  if (row > (int64_t)kNoAllocDoubles || n_tot > kNoAllocDoubles) {
    set_error("best_rminus1_noalloc: B*d + d + (blocks_S + blocks_M)*d*d + 2 = " + std::to_string(n_tot) +
              " doubles of scratch needed, the static array holds " + std::to_string(kNoAllocDoubles) +
              " (8 MiB; blocks_S = min(ceil(n*B/64), 592), blocks_M = min(ceil(B/64), 148)): use best_rminus1");
    return BEST_ERR_ARG;
  }
  double* buf = nullptr;
  BEST_TRY(noalloc_scratch(&buf));
  double *means = buf, *gm = means + n_means, *accS = gm + d, *accM = accS + (size_t)nblkS * dd,
         *out = accM + (size_t)nblkM * dd;
  k_chain_means<<<(unsigned)((row + 255) / 256), 256, 0, s>>>(trace_dev, n, row, means);
  k_grand_mean<<<1, 1024, 0, s>>>(means, B, d, gm);
  k_gram_partial<float><<<nblkS, G_TPB, 0, s>>>(trace_dev, n * B, d, gm, accS);
  k_gram_partial<double><<<nblkM, G_TPB, 0, s>>>(means, B, d, gm, accM);
  k_rminus1_finalize<<<1, 256, 0, s>>>(accS, nblkS, accM, nblkM, d, (double)n, (double)B, out);
  count_launch(5);
  double h[2] = {0.0, 0.0};
  if (cudaGetLastError() != cudaSuccess || cudaMemcpyAsync(h, out, sizeof(h), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
      cudaStreamSynchronize(s) != cudaSuccess) {
    set_error("best_rminus1_noalloc: CUDA failure");
    cudaGetLastError();
    return BEST_ERR_CUDA;
  }
  *rminus1_host = h[0];
  if (h[1] != 0.0) {
    set_error("best_rminus1_noalloc: the mean chain covariance is not positive definite (or some chain means coincide)");
    return BEST_ERR_NOT_SPD;
  }
  return BEST_OK;
}
