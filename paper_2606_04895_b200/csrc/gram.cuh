// Partial Gram sums in fp64 with a fixed summation order, shared by the covariance window of A9 (steps.cu)
// and the R - 1 diagnostic (diagnostics.cu).
#pragma once

#include "best_internal.h"

namespace best {

constexpr int G_TPB = 128;
constexpr int G_ROWS = 64;
// Position of column i inside a 32-double row of the SMEM tile: the first 16 slots hold the pairs (4t, 4t+1),
// t = 0..7, the last 16 the pairs (4t+2, 4t+3), so that the eight threads of a quarter-warp (t = 0..7) read one
// contiguous 128-byte run per 16-byte load (in natural order the 32-byte stride made these loads 2-way conflicted)
__host__ __device__ constexpr int gram_pos(int i) { return ((i & 2) << 3) | ((i >> 2) << 1) | (i & 1); }

// out[blk][i*d + j] = sum over the block's rows of (x_i - ref_i)(x_j - ref_j); rows are [nrows][d].
// The rows of a tile sit in SMEM padded to 32 columns (zeros); the 128 threads are two groups of 8 x 8
// threads, each thread holding a 4 x 4 block of the 32 x 32 Gram matrix in registers (two 32-byte SMEM
// reads, broadcast inside a warp, per 16 fp64 FMAs) and each group taking every other row of the tile.
template <typename T>
__global__ void __launch_bounds__(G_TPB)
k_gram_partial(const T* __restrict__ rows, int64_t nrows, int d, const double* __restrict__ ref,
               double* __restrict__ acc) {
  __shared__ __align__(16) double xs[G_ROWS * kMaxD];
  const int grp = threadIdx.x >> 6, u = threadIdx.x & 63, ti = u >> 3, tj = u & 7;
  double a4[4][4];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int q = 0; q < 4; ++q) a4[p][q] = 0.0;
  for (int e = threadIdx.x; e < G_ROWS * kMaxD; e += G_TPB) xs[e] = 0.0;   // the padding columns stay zero
  for (int64_t r0 = blockIdx.x * (int64_t)G_ROWS; r0 < nrows; r0 += (int64_t)gridDim.x * G_ROWS) {
    const int nv = (int)((nrows - r0 < G_ROWS) ? (nrows - r0) : G_ROWS);
    __syncthreads();
    {   // lane = column, warp = row (mod 4): 4 d-byte runs per instruction, no index division
      const int i = threadIdx.x & 31;
      if (i < d) {
        const double ri = ref[i];
        for (int r = threadIdx.x >> 5; r < G_ROWS; r += G_TPB / 32)
          xs[r * kMaxD + gram_pos(i)] = (r < nv) ? (double)rows[(r0 + r) * d + i] - ri : 0.0;
      }
    }
    __syncthreads();
    for (int r = grp; r < nv; r += 2) {
      const double2* pa = reinterpret_cast<const double2*>(xs + r * kMaxD) + ti;
      const double2* pb = reinterpret_cast<const double2*>(xs + r * kMaxD) + tj;
      const double2 a01 = pa[0], a23 = pa[8], b01 = pb[0], b23 = pb[8];
      const double a[4] = {a01.x, a01.y, a23.x, a23.y}, b[4] = {b01.x, b01.y, b23.x, b23.y};
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q) a4[p][q] = fma(a[p], b[q], a4[p][q]);
    }
  }
  // group 1 hands its block to group 0 through SMEM (fixed order: g0 + g1)
  __syncthreads();
  if (grp == 1)
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int q = 0; q < 4; ++q) xs[(4 * ti + p) * kMaxD + 4 * tj + q] = a4[p][q];
  __syncthreads();
  if (grp == 0)
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int i = 4 * ti + p, j = 4 * tj + q;
        if (i < d && j < d) acc[(size_t)blockIdx.x * d * d + i * d + j] = a4[p][q] + xs[i * kMaxD + j];
      }
}

// Covariance window of A9 fed in SEGMENTS: this launch adds the window's rows [row0, row0 + nrows) (global
// index inside the window; `rows` points at row row0) to running sums that live in global memory between
// launches.  The result does not depend on how the window was cut into segments: tile T = global rows
// [64 T, 64 T + 64) always belongs to block T mod gridDim.x and row parity picks the thread group, every
// thread CONTINUES its own running sums (loaded at the start, stored at the end), so each accumulator sees its
// rows in increasing global order whatever the segmentation.  The grid is fixed for the whole window.
// acc[(blk * 2 + grp) * ne + e], ne = 1 + d + d*d: e = 0 row count, 1..d sums of (x - ref), then products.
static __global__ void __launch_bounds__(G_TPB)
k_gram_window(const float* __restrict__ rows, int64_t row0, int64_t nrows, int d, const double* __restrict__ ref,
              double* __restrict__ acc) {
  __shared__ __align__(16) double xs[G_ROWS * kMaxD];
  const int grp = threadIdx.x >> 6, u = threadIdx.x & 63, ti = u >> 3, tj = u & 7;
  const int ne = 1 + d + d * d;
  double* mine = acc + ((size_t)blockIdx.x * 2 + grp) * ne;
  double a4[4][4], s4[4], cnt = 0.0;
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const int i = 4 * ti + p;
    s4[p] = (tj == 0 && i < d) ? mine[1 + i] : 0.0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int j = 4 * tj + q;
      a4[p][q] = (i < d && j < d) ? mine[1 + d + i * d + j] : 0.0;
    }
  }
  if (u == 0) cnt = mine[0];
  for (int e = threadIdx.x; e < G_ROWS * kMaxD; e += G_TPB) xs[e] = 0.0;   // the padding columns stay zero
  const int64_t rend = row0 + nrows;
  const int64_t t_first = row0 / G_ROWS, t_last = (rend - 1) / G_ROWS;
  int64_t T = t_first + (((int64_t)blockIdx.x - t_first % gridDim.x) + gridDim.x) % gridDim.x;   // first tile = blockIdx (mod grid)
  for (; T <= t_last; T += gridDim.x) {
    const int64_t g0 = T * G_ROWS;
    const int lo = (int)(g0 < row0 ? row0 - g0 : 0), hi = (int)(g0 + G_ROWS > rend ? rend - g0 : G_ROWS);   // rows [lo, hi) of the tile
    __syncthreads();
    {   // lane = column, warp = row (mod 4): 4 d-byte runs per instruction, no index division
      const int i = threadIdx.x & 31;
      if (i < d) {
        const double ri = ref[i];
        for (int r = lo + (threadIdx.x >> 5); r < hi; r += G_TPB / 32)
          xs[r * kMaxD + gram_pos(i)] = (double)rows[(g0 - row0 + r) * d + i] - ri;
      }
    }
    __syncthreads();
    for (int r = lo + ((lo ^ grp) & 1); r < hi; r += 2) {   // this group's parity
      const double2* pa = reinterpret_cast<const double2*>(xs + r * kMaxD) + ti;
      const double2* pb = reinterpret_cast<const double2*>(xs + r * kMaxD) + tj;
      const double2 a01 = pa[0], a23 = pa[8], b01 = pb[0], b23 = pb[8];
      const double a[4] = {a01.x, a01.y, a23.x, a23.y}, b[4] = {b01.x, b01.y, b23.x, b23.y};
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < 4; ++q) a4[p][q] = fma(a[p], b[q], a4[p][q]);
      if (tj == 0) {
#pragma unroll
        for (int p = 0; p < 4; ++p) s4[p] += a[p];
      }
      cnt += 1.0;
    }
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const int i = 4 * ti + p;
    if (tj == 0 && i < d) mine[1 + i] = s4[p];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int j = 4 * tj + q;
      if (i < d && j < d) mine[1 + d + i * d + j] = a4[p][q];
    }
  }
  if (u == 0) mine[0] = cnt;
}

}  // namespace best
