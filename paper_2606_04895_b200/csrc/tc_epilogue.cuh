// Epilogue / sampler side of the fused tensor-core kernel.  Included by tc_fused.cu only.
//
// 16 epilogue warps = 512 threads.  Thread (row, k): row = TMEM lane = chain, k = 0..3.
//   * MLP epilogues: of every 64-column group the thread handles columns [16k, 16k+16).
//   * sampler algebra: the thread owns parameter dimensions [8k, 8k+8) of its chain; the four
//     threads of a chain (same lane, four different warps of one TMEM lane quarter) exchange
//     matvec inputs and partial sums through SMEM with a 128-thread named barrier.
// Four resident warps per SM sub-partition hide the ALU / MUFU / LDS latencies that a single
// warp per sub-partition cannot.
#pragma once

namespace best {
namespace tc {

struct EpiCtx {
  const Params* P;
  Bars bars;
  uint8_t* smem;
  uint32_t tmem_lane;   // tmem base + (lane quarter << 16)
  int row;              // 0..127
  int k;                // 0..3
  uint32_t o, g;        // op / n-chunk counters (mirror the MMA issuer)
  uint32_t vslot, pslot;  // rotating scratch slots
  const float *bias_s, *wout_s, *wouts_s, *Ls, *LTs, *Rs, *RTs, *vecs;
  float* part;          // [2][4][128]
  uint16_t* dact_tile;
  // per-thread constants: byte offsets of this thread's two 16-B pieces inside an A k-chunk
  // (128B swizzle) and its element offset inside a [8 pieces][128 rows][8] act' block
  uint32_t a_off0, a_off1, dact_row_off;
};

using ptx::f32x2;

// address of 16-byte piece `p` of row `row` in A k-chunk `j` (128B swizzle)
__device__ __forceinline__ uint8_t* a_piece(const EpiCtx& C, int j, int p) {
  return C.smem + SmemLayout::A + j * kAChunkBytes + C.row * 128 + ((p ^ (C.row & 7)) << 4);
}
// act' scratch: [layer][chunk j][8 pieces][128 rows][8 bf16]; one (layer, j) block = 8192 elements
__device__ __forceinline__ uint16_t* dact_ptr(const EpiCtx& C, int layer, int j) {
  return C.dact_tile + (uint32_t)(layer * (C.P->H >> 6) + j) * 8192u + C.dact_row_off;
}
__device__ __forceinline__ uint8_t* a_chunk(const EpiCtx& C, int j) {
  return C.smem + SmemLayout::A + j * kAChunkBytes;
}
__device__ __forceinline__ void qbar(const EpiCtx& C) { ptx::named_bar_sync(1 + (C.row >> 5), 128); }

// ---- activations on fp32 pairs ---------------------------------------------------------------
// SiLU: h = a*sg, dact = sg + h*(1 - sg), sg = 1/(1 + 2^(-a log2 e)).
// kFastAct: sg = 0.5 + 0.5 tanh.approx(a/2)             (1 MUFU / element)
// else    : ex2.approx + bit-trick reciprocal + 2 Newton steps on the FMA pipe (1 MUFU / element,
//           relative error of sg ~2e-4, no cancellation for a << 0)
template <bool kFast>
__device__ __forceinline__ void silu2(f32x2 a, f32x2& h, f32x2& dact) {
  f32x2 sg;
  if (kFast) {
    float x0, x1;
    ptx::unpack2(ptx::mul2(a, ptx::pack2(0.5f, 0.5f)), x0, x1);
    const f32x2 t = ptx::pack2(ptx::tanh_approx(x0), ptx::tanh_approx(x1));
    sg = ptx::fma2(t, ptx::pack2(0.5f, 0.5f), ptx::pack2(0.5f, 0.5f));
  } else {
    float x0, x1;
    ptx::unpack2(ptx::mul2(a, ptx::pack2(-1.4426950408889634f, -1.4426950408889634f)), x0, x1);
    const f32x2 e = ptx::pack2(ptx::ex2_approx(fminf(x0, 80.0f)), ptx::ex2_approx(fminf(x1, 80.0f)));
    const f32x2 ns = ptx::fma2(e, ptx::pack2(-1.0f, -1.0f), ptx::pack2(-1.0f, -1.0f));  // -(1+e)
    uint32_t n0, n1;
    ptx::unpack2u(ns, n0, n1);
    f32x2 r = ptx::pack2u(0xFEF311C7u - n0, 0xFEF311C7u - n1);   // ~1/(1+e), 12 % accurate
    const f32x2 two = ptx::pack2(2.0f, 2.0f);
    r = ptx::mul2(r, ptx::fma2(ns, r, two));
    r = ptx::mul2(r, ptx::fma2(ns, r, two));
    sg = r;
  }
  h = ptx::mul2(a, sg);
  const f32x2 omr = ptx::fma2(sg, ptx::pack2(-1.0f, -1.0f), ptx::pack2(1.0f, 1.0f));
  dact = ptx::fma2(h, omr, sg);
}
__device__ __forceinline__ void tanh2(f32x2 a, f32x2& h, f32x2& dact) {
  float x0, x1;
  ptx::unpack2(a, x0, x1);
  h = ptx::pack2(ptx::tanh_approx(x0), ptx::tanh_approx(x1));
  dact = ptx::fma2(ptx::mul2(h, h), ptx::pack2(-1.0f, -1.0f), ptx::pack2(1.0f, 1.0f));
}

#ifndef BEST_TC_FAST_ACT
#define BEST_TC_FAST_ACT 0
#endif

// ---- first A operand: theta split into bf16 hi | lo (own 8 dims -> pieces k and 4+k) ------------
__device__ __forceinline__ void write_xin(EpiCtx& C, const float (&th)[8]) {
  ptx::mbar_wait(C.bars.a_free(0), (C.o & 1u) ^ 1u);
  uint32_t hi[4], lo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t h2 = ptx::pack_bf16x2(th[2 * i], th[2 * i + 1]);
    hi[i] = h2;
    lo[i] = ptx::pack_bf16x2(th[2 * i] - ptx::bf16_lo(h2), th[2 * i + 1] - ptx::bf16_hi(h2));
  }
  *reinterpret_cast<uint4*>(a_piece(C, 0, C.k)) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
  *reinterpret_cast<uint4*>(a_piece(C, 0, 4 + C.k)) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  ptx::fence_proxy_async();
#pragma unroll
  for (int j = 0; j < kMaxKch; ++j) ptx::mbar_arrive(C.bars.a_ready(j));
}

// forward epilogue of one op: bias + activation (+ act' to scratch, or delta for the last layer)
template <int ACT, bool LAST>
__device__ __forceinline__ void epi_fwd(EpiCtx& C, const OpDesc& op, bool want_grad, float& acc_out,
                                        int& written) {
  const Params& P = *C.P;
  const bool writes_a = !(LAST && !want_grad);
  for (int c = 0; c < op.nch; ++c, ++C.g) {
    const uint32_t buf = C.g & 1u, use = C.g >> 1;
    ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
    ptx::tc_fence_after();
    const uint32_t tcol = C.tmem_lane + buf * 256u + C.k * 16;
    const int ngrp = op.ncols / 64;
    for (int grp = 0; grp < ngrp; ++grp) {
      const int jn = (c * op.ncols) / 64 + grp;
      uint32_t v[16];
      ptx::tmem_ld16(tcol + grp * 64, v);
      const int f0 = jn * 64 + C.k * 16;
      const float* bp = C.bias_s + op.layer * P.H + f0;
      if (writes_a) ptx::mbar_wait(C.bars.a_free(jn), C.o & 1u);
      ptx::tmem_ld_wait();
      uint32_t hp[8], dp[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float2 b = *reinterpret_cast<const float2*>(bp + 2 * i);
        const f32x2 a = ptx::add2(ptx::pack2u(v[2 * i], v[2 * i + 1]), ptx::pack2(b.x, b.y));
        f32x2 h, dd;
        if (ACT == BEST_ACT_SILU) silu2<BEST_TC_FAST_ACT != 0>(a, h, dd); else tanh2(a, h, dd);
        if (LAST) {
          const float2 w = *reinterpret_cast<const float2*>(C.wout_s + f0 + 2 * i);
          float h0, h1;
          ptx::unpack2(h, h0, h1);
          acc_out = fmaf(h0, w.x, acc_out);
          acc_out = fmaf(h1, w.y, acc_out);
          if (want_grad) {
            const float2 ws = *reinterpret_cast<const float2*>(C.wouts_s + f0 + 2 * i);
            hp[i] = ptx::pack_bf16x2_from(ptx::mul2(dd, ptx::pack2(ws.x, ws.y)));
          }
        } else {
          hp[i] = ptx::pack_bf16x2_from(h);
          dp[i] = ptx::pack_bf16x2_from(dd);
        }
      }
      if (!LAST && want_grad) {
        uint16_t* dptr = dact_ptr(C, op.layer, jn);
        *reinterpret_cast<uint4*>(dptr) = make_uint4(dp[0], dp[1], dp[2], dp[3]);
        *reinterpret_cast<uint4*>(dptr + 1024) = make_uint4(dp[4], dp[5], dp[6], dp[7]);
      }
      if (writes_a) {
        uint8_t* ach = a_chunk(C, jn);
        *reinterpret_cast<uint4*>(ach + C.a_off0) = make_uint4(hp[0], hp[1], hp[2], hp[3]);
        *reinterpret_cast<uint4*>(ach + C.a_off1) = make_uint4(hp[4], hp[5], hp[6], hp[7]);
        ptx::fence_proxy_async();
        ptx::mbar_arrive(C.bars.a_ready(jn));
        written = jn + 1;
      }
    }
    ptx::tc_fence_before();
    ptx::mbar_arrive(C.bars.d_free(buf));
  }
}

// backward epilogue: delta_{l-1} = (delta_l W_l) .* act'_{l-1}
__device__ __forceinline__ void epi_bwd(EpiCtx& C, const OpDesc& op, int& written) {
  const Params& P = *C.P;
  for (int c = 0; c < op.nch; ++c, ++C.g) {
    const uint32_t buf = C.g & 1u, use = C.g >> 1;
    ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
    ptx::tc_fence_after();
    const uint32_t tcol = C.tmem_lane + buf * 256u + C.k * 16;
    const int ngrp = op.ncols / 64;
    for (int grp = 0; grp < ngrp; ++grp) {
      const int jn = (c * op.ncols) / 64 + grp;
      uint32_t v[16];
      ptx::tmem_ld16(tcol + grp * 64, v);
      const uint16_t* dptr = dact_ptr(C, op.layer, jn);
      const uint4 d0 = *reinterpret_cast<const uint4*>(dptr);
      const uint4 d1 = *reinterpret_cast<const uint4*>(dptr + 1024);
      const uint32_t dw[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
      ptx::mbar_wait(C.bars.a_free(jn), C.o & 1u);
      ptx::tmem_ld_wait();
      uint32_t hp[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const f32x2 dd = ptx::pack2u(dw[i] << 16, dw[i] & 0xFFFF0000u);
        hp[i] = ptx::pack_bf16x2_from(ptx::mul2(ptx::pack2u(v[2 * i], v[2 * i + 1]), dd));
      }
      uint8_t* ach = a_chunk(C, jn);
      *reinterpret_cast<uint4*>(ach + C.a_off0) = make_uint4(hp[0], hp[1], hp[2], hp[3]);
      *reinterpret_cast<uint4*>(ach + C.a_off1) = make_uint4(hp[4], hp[5], hp[6], hp[7]);
      ptx::fence_proxy_async();
      ptx::mbar_arrive(C.bars.a_ready(jn));
      written = jn + 1;
    }
    ptx::tc_fence_before();
    ptx::mbar_arrive(C.bars.d_free(buf));
  }
}

// One MLP evaluation.  In: own 8 dims of theta.  Out: this thread's PARTIAL of the MLP output sum
// (over its columns) and, when want_grad, s * d MLP / d theta for its own 8 dims.
__device__ __forceinline__ void tc_eval(EpiCtx& C, const float (&th)[8], bool want_grad, float& out_part,
                                        float (&gm)[8]) {
  const Params& P = *C.P;
  write_xin(C, th);
  float acc_out = 0.0f;
  const int n_ops = want_grad ? P.n_ops_all : P.n_ops_fwd;
  for (int oi = 0; oi < n_ops; ++oi, ++C.o) {
    const OpDesc op = P.ops[oi];
    int written = 0;
    if (op.epi == EPI_FWD_HID) {
      if (P.act == BEST_ACT_SILU) epi_fwd<BEST_ACT_SILU, false>(C, op, want_grad, acc_out, written);
      else epi_fwd<BEST_ACT_TANH, false>(C, op, want_grad, acc_out, written);
    } else if (op.epi == EPI_FWD_LAST) {
      if (P.act == BEST_ACT_SILU) epi_fwd<BEST_ACT_SILU, true>(C, op, want_grad, acc_out, written);
      else epi_fwd<BEST_ACT_TANH, true>(C, op, want_grad, acc_out, written);
    } else if (op.epi == EPI_BWD_HID) {
      epi_bwd(C, op, written);
    } else {  // EPI_BWD_FINAL: D[128][32] -> own 8 columns
      const uint32_t buf = C.g & 1u, use = C.g >> 1;
      ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
      ptx::tc_fence_after();
      uint32_t v[8];
      ptx::tmem_ld8(C.tmem_lane + buf * 256u + C.k * 8, v);
      ptx::tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 8; ++i) gm[i] = __uint_as_float(v[i]);
      ptx::tc_fence_before();
      ptx::mbar_arrive(C.bars.d_free(buf));
      ++C.g;
    }
    if (oi != n_ops - 1)  // keep every a_ready barrier at one phase per op
      for (int j = written; j < kMaxKch; ++j) ptx::mbar_arrive(C.bars.a_ready(j));
  }
  out_part = acc_out;
}

// ---- cooperative per-chain algebra: each thread owns dims [8k, 8k+8) ---------------------------
__device__ __forceinline__ float* vslot_ptr(EpiCtx& C) {   // rotate between A chunks 1 and 2
  C.vslot ^= 1u;
  return reinterpret_cast<float*>(C.smem + SmemLayout::A + (1 + C.vslot) * kAChunkBytes);
}
__device__ __forceinline__ const float* share(EpiCtx& C, const float (&x)[8]) {
  float* V = vslot_ptr(C);
#pragma unroll
  for (int i = 0; i < 8; ++i) V[(8 * C.k + i) * kRows + C.row] = x[i];
  qbar(C);
  return V;
}
// out[i] = sum_{j in [j0, j1)} M[j*32 + 8k + i] * V[j]   (M row j holds the 8 coefficients contiguously)
__device__ __forceinline__ void mv_rows(const EpiCtx& C, const float* __restrict__ M, const float* V, int j0,
                                        int j1, float (&out)[8]) {
#pragma unroll
  for (int i = 0; i < 8; ++i) out[i] = 0.0f;
  for (int j = j0; j < j1; ++j) {
    const float vj = V[j * kRows + C.row];
    const float4 m0 = *reinterpret_cast<const float4*>(M + j * kDP + 8 * C.k);
    const float4 m1 = *reinterpret_cast<const float4*>(M + j * kDP + 8 * C.k + 4);
    out[0] = fmaf(m0.x, vj, out[0]); out[1] = fmaf(m0.y, vj, out[1]);
    out[2] = fmaf(m0.z, vj, out[2]); out[3] = fmaf(m0.w, vj, out[3]);
    out[4] = fmaf(m1.x, vj, out[4]); out[5] = fmaf(m1.y, vj, out[5]);
    out[6] = fmaf(m1.z, vj, out[6]); out[7] = fmaf(m1.w, vj, out[7]);
  }
}
// out = L x : out_i = sum_{j<=i} L[i][j] x_j, own i  -> coefficients LT[j][i], j in [0, 8k+8)
__device__ __forceinline__ void mv_L(EpiCtx& C, const float (&x)[8], float (&out)[8]) {
  const float* V = share(C, x);
  mv_rows(C, C.LTs, V, 0, 8 * C.k + 8, out);
}
// out = L^T x : out_j = sum_{i>=j} L[i][j] x_i, own j -> coefficients L[i][j], i in [8k, 32)
__device__ __forceinline__ void mv_Lt(EpiCtx& C, const float (&x)[8], float (&out)[8]) {
  const float* V = share(C, x);
  mv_rows(C, C.Ls, V, 8 * C.k, kDP, out);
}
__device__ __forceinline__ float reduce4(EpiCtx& C, float x) {
  C.pslot ^= 1u;
  float* Pp = C.part + C.pslot * 4 * kRows;
  Pp[C.k * kRows + C.row] = x;
  qbar(C);
  return (Pp[C.row] + Pp[kRows + C.row]) + (Pp[2 * kRows + C.row] + Pp[3 * kRows + C.row]);
}

// full target from the MLP partial output + Gaussian (y = R r), banana and box terms.
// lp is identical on the four threads of a chain; g covers the thread's own 8 dims.
__device__ __forceinline__ void finish_target(EpiCtx& C, const float (&th)[8], float out_part, bool want_grad,
                                              float& lp, float (&g)[8]) {
  const Params& P = *C.P;
  float part = P.mlp_scale * out_part;
  float ti = 0.0f, tj = 0.0f;
  if (P.has_gauss || P.banana_i >= 0) {
    float r[8], y[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) r[i] = th[i] - C.vecs[8 * C.k + i];
    const float* V = share(C, r);
    if (P.banana_i >= 0) {
      ti = V[P.banana_i * kRows + C.row] + C.vecs[P.banana_i];
      tj = V[P.banana_j * kRows + C.row] + C.vecs[P.banana_j];
    }
    if (P.has_gauss) {
      mv_rows(C, C.RTs, V, 8 * C.k, kDP, y);          // y_i = sum_{j>=i} R[i][j] r_j
#pragma unroll
      for (int i = 0; i < 8; ++i) part = fmaf(-0.5f * y[i], y[i], part);
      if (want_grad) {
        float gg[8];
        const float* Vy = share(C, y);
        mv_rows(C, C.Rs, Vy, 0, 8 * C.k + 8, gg);      // (R^T y)_j = sum_{i<=j} R[i][j] y_i
#pragma unroll
        for (int i = 0; i < 8; ++i) g[i] -= gg[i];
      }
    }
  }
  if (P.has_box) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int gi = 8 * C.k + i;
      const float lo = C.vecs[32 + gi], hi = C.vecs[64 + gi], iw = C.vecs[96 + gi];
      const float ex = fmaxf(fmaxf(lo - th[i], th[i] - hi), 0.0f);
      if (ex > 0.0f) {
        const float t = P.pen_gamma * ex * iw;
        float f, df;
        if (t <= 40.0f) { df = expm1f(t); f = df - t; }
        else { df = 2.3538526683701998e17f; f = (df - 40.0f) + df * (t - 40.0f); }
        part -= P.pen_kappa * f;
        g[i] -= P.pen_kappa * df * P.pen_gamma * iw * ((th[i] > hi) ? 1.0f : -1.0f);
      }
    }
  }
  lp = reduce4(C, part) + P.mlp_scale * P.b_out;
  if (P.banana_i >= 0) {
    const float t = tj - ti * ti, inv = 1.0f / (P.banana_sigma * P.banana_sigma);
    lp -= 0.5f * t * t * inv;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (8 * C.k + i == P.banana_j) g[i] -= t * inv;
      if (8 * C.k + i == P.banana_i) g[i] += 2.0f * ti * t * inv;
    }
  }
}

// evaluate the full target at th (own dims): lp (same on all 4 threads) and own 8 gradient dims
__device__ __forceinline__ void eval_target(EpiCtx& C, const float (&th)[8], bool want_grad, float& lp,
                                            float (&g)[8]) {
  float out_part;
#pragma unroll
  for (int i = 0; i < 8; ++i) g[i] = 0.0f;
  tc_eval(C, th, want_grad, out_part, g);
  finish_target(C, th, out_part, want_grad, lp, g);
}

// own 8 normals: Philox blocks 2k and 2k+1 (slot 1+j -> dims 4j..4j+3)
__device__ __forceinline__ void draw_normals8(const EpiCtx& C, uint64_t seed, uint32_t chain, uint64_t step,
                                              int d, float (&xi)[8]) {
#pragma unroll
  for (int b = 0; b < 2; ++b) {
    const int j = 2 * C.k + b;
    if (4 * j < d) {
      const uint4 w = philox4x32_10(chain, step, (uint32_t)(1 + j), seed);
      box_muller(w.x, w.y, xi[4 * b], xi[4 * b + 1]);
      box_muller(w.z, w.w, xi[4 * b + 2], xi[4 * b + 3]);
    } else {
      xi[4 * b] = xi[4 * b + 1] = xi[4 * b + 2] = xi[4 * b + 3] = 0.0f;
    }
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) if (8 * C.k + i >= d) xi[i] = 0.0f;
}

__device__ __forceinline__ void load_vec8(const EpiCtx& C, const double* a, int64_t ld, int64_t c, int d,
                                          bool valid, float (&v)[8]) {
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int gi = 8 * C.k + i;
    v[i] = (valid && gi < d) ? (float)a[(int64_t)gi * ld + c] : 0.0f;
  }
}
__device__ __forceinline__ void store_vec8(const EpiCtx& C, double* a, int64_t ld, int64_t c, int d,
                                           const float (&v)[8]) {
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int gi = 8 * C.k + i;
    if (gi < d) a[(int64_t)gi * ld + c] = (double)v[i];
  }
}

}  // namespace tc
}  // namespace best
