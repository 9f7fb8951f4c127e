// Device-side RNG and per-chain algebra shared by the step kernels (fp64 on the exact path,
// fp32 inside the tensor-core kernel).  Written from the paper + DESIGN.md readings; shares
// nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace best {

// Philox4x32-10 (Salmon et al., SC'11).  north_star: RNG keyed by (seed, chain, step).
// counter = (chain, step lo, step hi, slot); key = (seed lo, seed hi)   [reading R1]
__device__ __forceinline__ uint4 philox4x32_10(uint32_t chain, uint64_t step, uint32_t slot,
                                               uint64_t seed) {
  uint32_t c0 = chain, c1 = (uint32_t)step, c2 = (uint32_t)(step >> 32), c3 = slot;
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

// u = ((x >> 9) + 0.5) * 2^-23: exact in fp32 and fp64, never 0 or 1   [reading R2]
template <typename real>
__device__ __forceinline__ real u01(uint32_t x) {
  return ((real)(x >> 9) + (real)0.5) * (real)(1.0 / 8388608.0);
}

// Box–Muller pair   [reading R3]
__device__ __forceinline__ void box_muller(uint32_t w0, uint32_t w1, double& n0, double& n1) {
  const double u1 = u01<double>(w0), u2 = u01<double>(w1);
  const double r = sqrt(-2.0 * log(u1));
  double s, c;
  sincospi(2.0 * u2, &s, &c);
  n0 = r * c;
  n1 = r * s;
}
__device__ __forceinline__ void box_muller(uint32_t w0, uint32_t w1, float& n0, float& n1) {
  const float u1 = u01<float>(w0), u2 = u01<float>(w1);
  const float r = sqrtf(-2.0f * logf(u1));
  float s, c;
  sincospif(2.0f * u2, &s, &c);
  n0 = r * c;
  n1 = r * s;
}

// slot 1+j -> normals of dims 4j..4j+3.  xi must have room for 4*ceil(d/4) values.
template <typename real>
__device__ __forceinline__ void draw_normals(uint64_t seed, uint32_t chain, uint64_t step, int d,
                                             real* xi) {
  const int nblk = (d + 3) >> 2;
  for (int j = 0; j < nblk; ++j) {
    const uint4 w = philox4x32_10(chain, step, (uint32_t)(1 + j), seed);
    box_muller(w.x, w.y, xi[4 * j + 0], xi[4 * j + 1]);
    box_muller(w.z, w.w, xi[4 * j + 2], xi[4 * j + 3]);
  }
}

// Accept rule (reading R7): accept iff log u < log alpha; NaN -> false.
template <typename real>
__device__ __forceinline__ bool accept_rule(real u, real log_alpha) {
  return log(u) < log_alpha;
}
template <>
__device__ __forceinline__ bool accept_rule<float>(float u, float log_alpha) {
  return logf(u) < log_alpha;
}

// out = L v (L lower triangular row-major [d][d])
template <typename real>
__device__ __forceinline__ void tri_L_apply(const double* __restrict__ L, int d, const real* v,
                                            real* out) {
  for (int i = 0; i < d; ++i) {
    real s = 0;
    for (int j = 0; j <= i; ++j) s += (real)L[i * d + j] * v[j];
    out[i] = s;
  }
}
// out = L^T v
template <typename real>
__device__ __forceinline__ void tri_Lt_apply(const double* __restrict__ L, int d, const real* v,
                                             real* out) {
  for (int j = 0; j < d; ++j) {
    real s = 0;
    for (int i = j; i < d; ++i) s += (real)L[i * d + j] * v[i];
    out[j] = s;
  }
}

}  // namespace best
