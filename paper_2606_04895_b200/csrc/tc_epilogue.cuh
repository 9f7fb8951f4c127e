// Epilogue / sampler side of the fused tensor-core kernel: one thread per chain (TMEM lane).
// Included by tc_fused.cu only.
#pragma once

namespace best {
namespace tc {

struct EpiCtx {
  const Params* P;
  Bars bars;
  uint8_t* smem;        // generic pointer to the dynamic smem base
  uint32_t tmem_lane;   // tmem base + (lane quarter << 16)
  int row;              // 0..127
  uint32_t o, g;        // op / n-chunk counters (mirror the MMA issuer)
  const float *bias_s, *wout_s, *wouts_s, *Ls, *Rs, *vecs;
  uint16_t* dact_tile;  // this CTA's act' scratch
};

// h = act(a), dact = act'(a).  One MUFU.EX2 + one MUFU.RCP per element, ~fp32 accurate.
__device__ __forceinline__ void act_eval(int kind, float a, float& h, float& dact) {
  if (kind == BEST_ACT_SILU) {
    const float e = ptx::ex2_approx(-1.4426950408889634f * fabsf(a));
    const float r = ptx::rcp_approx(1.0f + e);
    const float sg = (a >= 0.0f) ? r : e * r;
    h = a * sg;
    dact = fmaf(h, 1.0f - sg, sg);
  } else {
    const float e = ptx::ex2_approx(-2.8853900817779268f * fabsf(a));
    const float t = (1.0f - e) * ptx::rcp_approx(1.0f + e);
    h = copysignf(t, a);
    dact = fmaf(-h, h, 1.0f);
  }
}

__device__ __forceinline__ void st_shared_v4(uint8_t* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  *reinterpret_cast<uint4*>(p) = make_uint4(a, b, c, d);
}

// address of 16-byte piece `p` of row `row` in A k-chunk `j` (128B swizzle)
__device__ __forceinline__ uint8_t* a_piece(const EpiCtx& C, int j, int p) {
  return C.smem + SmemLayout::A + j * kAChunkBytes + C.row * 128 + ((p ^ (C.row & 7)) << 4);
}

__device__ __forceinline__ size_t dact_off(const Params& P, int layer, int j, int p, int row) {
  return ((((size_t)layer * (P.H / 64) + j) * 8 + p) * kRows + row) * 8;
}

// The first A operand of an evaluation: theta split into bf16 hi | lo halves (K = 64), so the
// input layer sees ~16 mantissa bits of theta although the MMA operands are bf16.
__device__ __forceinline__ void write_xin(EpiCtx& C, const float (&th)[kDP]) {
  ptx::mbar_wait(C.bars.a_free[0], (C.o & 1u) ^ 1u);  // previous op has finished reading chunk 0
  uint32_t hi[16], lo[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const uint32_t h2 = ptx::pack_bf16x2(th[2 * i], th[2 * i + 1]);
    hi[i] = h2;
    lo[i] = ptx::pack_bf16x2(th[2 * i] - ptx::bf16_lo(h2), th[2 * i + 1] - ptx::bf16_hi(h2));
  }
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    st_shared_v4(a_piece(C, 0, p), hi[4 * p], hi[4 * p + 1], hi[4 * p + 2], hi[4 * p + 3]);
    st_shared_v4(a_piece(C, 0, 4 + p), lo[4 * p], lo[4 * p + 1], lo[4 * p + 2], lo[4 * p + 3]);
  }
  ptx::fence_proxy_async();
#pragma unroll
  for (int j = 0; j < kMaxKch; ++j) ptx::mbar_arrive(C.bars.a_ready[j]);
}

// One MLP evaluation for this thread's chain: forward (and input-gradient when want_grad).
// Returns the raw MLP output and d out / d theta (unscaled by s? no: gm already carries s).
__device__ __forceinline__ void tc_eval(EpiCtx& C, const float (&th)[kDP], bool want_grad, float& out,
                                        float (&gm)[kDP]) {
  const Params& P = *C.P;
  write_xin(C, th);
  float acc_out = 0.0f;
  const int n_ops = want_grad ? P.n_ops_all : P.n_ops_fwd;
  for (int oi = 0; oi < n_ops; ++oi, ++C.o) {
    const OpDesc op = P.ops[oi];
    const bool last_op = (oi == n_ops - 1);
    int written = 0;
    for (int c = 0; c < op.nch; ++c, ++C.g) {
      const uint32_t buf = C.g & 1u, use = C.g >> 1;
      ptx::mbar_wait(C.bars.d_full[buf], use & 1u);
      ptx::tc_fence_after();
      const uint32_t tcol = C.tmem_lane + buf * 256u;
      if (op.epi == EPI_BWD_FINAL) {
        uint32_t v[32];
        ptx::tmem_ld32(tcol, v);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < kDP; ++i) gm[i] = __uint_as_float(v[i]);
      } else {
        const int ngrp = op.ncols / 64;
        for (int grp = 0; grp < ngrp; ++grp) {
          const int jn = (c * op.ncols) / 64 + grp;  // A' chunk produced by these 64 columns
          const bool writes_a = !(op.epi == EPI_FWD_LAST && !want_grad);
          if (writes_a) ptx::mbar_wait(C.bars.a_free[jn], C.o & 1u);
#pragma unroll
          for (int half = 0; half < 2; ++half) {
            uint32_t v[32];
            ptx::tmem_ld32(tcol + grp * 64 + half * 32, v);
            const int f0 = jn * 64 + half * 32;  // feature index of v[0]
            uint4 dl[4];
            if (op.epi == EPI_BWD_HID) {
#pragma unroll
              for (int q = 0; q < 4; ++q)
                dl[q] = *reinterpret_cast<const uint4*>(C.dact_tile +
                                                        dact_off(P, op.layer, jn, half * 4 + q, C.row));
            }
            ptx::tmem_ld_wait();
#pragma unroll
            for (int q = 0; q < 4; ++q) {
              uint32_t hp[4], dp[4];
              if (op.epi == EPI_BWD_HID) {
                const uint32_t dw[4] = {dl[q].x, dl[q].y, dl[q].z, dl[q].w};
#pragma unroll
                for (int e2 = 0; e2 < 4; ++e2) {
                  const float x0 = __uint_as_float(v[q * 8 + 2 * e2]) * ptx::bf16_lo(dw[e2]);
                  const float x1 = __uint_as_float(v[q * 8 + 2 * e2 + 1]) * ptx::bf16_hi(dw[e2]);
                  hp[e2] = ptx::pack_bf16x2(x0, x1);
                }
              } else {
                const float4 b0 = *reinterpret_cast<const float4*>(C.bias_s + op.layer * P.H + f0 + q * 8);
                const float4 b1 = *reinterpret_cast<const float4*>(C.bias_s + op.layer * P.H + f0 + q * 8 + 4);
                const float bb[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
                float hh[8], dd[8];
#pragma unroll
                for (int e = 0; e < 8; ++e)
                  act_eval(P.act, __uint_as_float(v[q * 8 + e]) + bb[e], hh[e], dd[e]);
                if (op.epi == EPI_FWD_LAST) {
                  const float4 w0 = *reinterpret_cast<const float4*>(C.wout_s + f0 + q * 8);
                  const float4 w1 = *reinterpret_cast<const float4*>(C.wout_s + f0 + q * 8 + 4);
                  const float ww[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
                  for (int e = 0; e < 8; ++e) acc_out = fmaf(hh[e], ww[e], acc_out);
                  if (want_grad) {
                    const float4 s0 = *reinterpret_cast<const float4*>(C.wouts_s + f0 + q * 8);
                    const float4 s1 = *reinterpret_cast<const float4*>(C.wouts_s + f0 + q * 8 + 4);
                    const float ss[8] = {s0.x, s0.y, s0.z, s0.w, s1.x, s1.y, s1.z, s1.w};
#pragma unroll
                    for (int e2 = 0; e2 < 4; ++e2)
                      hp[e2] = ptx::pack_bf16x2(ss[2 * e2] * dd[2 * e2], ss[2 * e2 + 1] * dd[2 * e2 + 1]);
                  }
                } else {
#pragma unroll
                  for (int e2 = 0; e2 < 4; ++e2) {
                    hp[e2] = ptx::pack_bf16x2(hh[2 * e2], hh[2 * e2 + 1]);
                    dp[e2] = ptx::pack_bf16x2(dd[2 * e2], dd[2 * e2 + 1]);
                  }
                  if (want_grad)
                    *reinterpret_cast<uint4*>(C.dact_tile + dact_off(P, op.layer, jn, half * 4 + q, C.row)) =
                        make_uint4(dp[0], dp[1], dp[2], dp[3]);
                }
              }
              if (writes_a) st_shared_v4(a_piece(C, jn, half * 4 + q), hp[0], hp[1], hp[2], hp[3]);
            }
          }
          if (writes_a) {
            ptx::fence_proxy_async();
            ptx::mbar_arrive(C.bars.a_ready[jn]);
            written = jn + 1;
          }
        }
      }
      ptx::tc_fence_before();
      ptx::mbar_arrive(C.bars.d_free[buf]);
    }
    if (!last_op)  // keep every a_ready barrier at one phase per op
      for (int j = written; j < kMaxKch; ++j) ptx::mbar_arrive(C.bars.a_ready[j]);
  }
  out = acc_out + P.b_out;
}

// ---- per-chain algebra in fp32 (vectors padded to 32, matrices zero padded in SMEM) -------------
__device__ __forceinline__ void mv_L(const float* __restrict__ Ls, const float (&v)[kDP], float (&out)[kDP]) {
#pragma unroll
  for (int i = 0; i < kDP; ++i) {
    float s = 0.0f;
#pragma unroll
    for (int j4 = 0; j4 <= i / 4; ++j4) {
      const float4 l = *reinterpret_cast<const float4*>(Ls + i * kDP + j4 * 4);
      s = fmaf(l.x, v[j4 * 4], s); s = fmaf(l.y, v[j4 * 4 + 1], s);
      s = fmaf(l.z, v[j4 * 4 + 2], s); s = fmaf(l.w, v[j4 * 4 + 3], s);
    }
    out[i] = s;
  }
}
__device__ __forceinline__ void mv_Lt(const float* __restrict__ Ls, const float (&v)[kDP], float (&out)[kDP]) {
#pragma unroll
  for (int j = 0; j < kDP; ++j) out[j] = 0.0f;
#pragma unroll
  for (int i = 0; i < kDP; ++i) {
#pragma unroll
    for (int j4 = 0; j4 <= i / 4; ++j4) {
      const float4 l = *reinterpret_cast<const float4*>(Ls + i * kDP + j4 * 4);
      out[j4 * 4] = fmaf(l.x, v[i], out[j4 * 4]); out[j4 * 4 + 1] = fmaf(l.y, v[i], out[j4 * 4 + 1]);
      out[j4 * 4 + 2] = fmaf(l.z, v[i], out[j4 * 4 + 2]); out[j4 * 4 + 3] = fmaf(l.w, v[i], out[j4 * 4 + 3]);
    }
  }
}

// log pi(theta) and gradient from the MLP output (already scaled by s in gm) + the cheap terms.
__device__ __forceinline__ void finish_target(const EpiCtx& C, const float (&th)[kDP], float mlp_out,
                                              bool want_grad, float& lp, float (&g)[kDP]) {
  const Params& P = *C.P;
  lp = P.mlp_scale * mlp_out;
  if (P.has_gauss) {  // y = R r (R upper triangular), logp -= |y|^2/2, g -= R^T y
    float r[kDP], y[kDP];
#pragma unroll
    for (int i = 0; i < kDP; ++i) r[i] = th[i] - C.vecs[i];
    float q = 0.0f;
#pragma unroll
    for (int i = 0; i < kDP; ++i) {
      float s = 0.0f;
#pragma unroll
      for (int j4 = i / 4; j4 < kDP / 4; ++j4) {
        const float4 l = *reinterpret_cast<const float4*>(C.Rs + i * kDP + j4 * 4);
        s = fmaf(l.x, r[j4 * 4], s); s = fmaf(l.y, r[j4 * 4 + 1], s);
        s = fmaf(l.z, r[j4 * 4 + 2], s); s = fmaf(l.w, r[j4 * 4 + 3], s);
      }
      y[i] = s;
      q = fmaf(s, s, q);
    }
    lp -= 0.5f * q;
    if (want_grad) {
#pragma unroll
      for (int i = 0; i < kDP; ++i) {
#pragma unroll
        for (int j4 = i / 4; j4 < kDP / 4; ++j4) {
          const float4 l = *reinterpret_cast<const float4*>(C.Rs + i * kDP + j4 * 4);
          g[j4 * 4] = fmaf(-l.x, y[i], g[j4 * 4]); g[j4 * 4 + 1] = fmaf(-l.y, y[i], g[j4 * 4 + 1]);
          g[j4 * 4 + 2] = fmaf(-l.z, y[i], g[j4 * 4 + 2]); g[j4 * 4 + 3] = fmaf(-l.w, y[i], g[j4 * 4 + 3]);
        }
      }
    }
  }
  if (P.banana_i >= 0) {
    float ti = 0.f, tj = 0.f;
#pragma unroll
    for (int i = 0; i < kDP; ++i) { if (i == P.banana_i) ti = th[i]; if (i == P.banana_j) tj = th[i]; }
    const float t = tj - ti * ti, inv = 1.0f / (P.banana_sigma * P.banana_sigma);
    lp -= 0.5f * t * t * inv;
#pragma unroll
    for (int i = 0; i < kDP; ++i) {
      if (i == P.banana_j) g[i] -= t * inv;
      if (i == P.banana_i) g[i] += 2.0f * ti * t * inv;
    }
  }
  if (P.has_box) {
    float pen = 0.0f;
#pragma unroll
    for (int i = 0; i < kDP; ++i) {
      const float lo = C.vecs[32 + i], hi = C.vecs[64 + i], iw = C.vecs[96 + i];
      const float ex = fmaxf(fmaxf(lo - th[i], th[i] - hi), 0.0f);
      if (ex > 0.0f) {
        const float t = P.pen_gamma * ex * iw;
        float f, df;
        if (t <= 40.0f) { df = expm1f(t); f = df - t; }
        else { df = 2.3538526683701998e17f; f = (df - 40.0f) + df * (t - 40.0f); }
        pen += f;
        g[i] -= P.pen_kappa * df * P.pen_gamma * iw * ((th[i] > hi) ? 1.0f : -1.0f);
      }
    }
    lp -= P.pen_kappa * pen;
  }
}

__device__ __forceinline__ void draw_normals32(uint64_t seed, uint32_t chain, uint64_t step, int d,
                                               float (&xi)[kDP]) {
  const int nblk = (d + 3) >> 2;
#pragma unroll
  for (int j = 0; j < kDP / 4; ++j) {
    if (j < nblk) {
      const uint4 w = philox4x32_10(chain, step, (uint32_t)(1 + j), seed);
      box_muller(w.x, w.y, xi[4 * j], xi[4 * j + 1]);
      box_muller(w.z, w.w, xi[4 * j + 2], xi[4 * j + 3]);
    } else {
      xi[4 * j] = xi[4 * j + 1] = xi[4 * j + 2] = xi[4 * j + 3] = 0.0f;
    }
  }
#pragma unroll
  for (int i = 0; i < kDP; ++i) if (i >= d) xi[i] = 0.0f;
}

__device__ __forceinline__ void load_vec(const double* a, int64_t ld, int64_t c, int d, bool valid,
                                         float (&v)[kDP]) {
#pragma unroll
  for (int i = 0; i < kDP; ++i) v[i] = (valid && i < d) ? (float)a[i * ld + c] : 0.0f;
}
__device__ __forceinline__ void store_vec(double* a, int64_t ld, int64_t c, int d, const float (&v)[kDP]) {
#pragma unroll
  for (int i = 0; i < kDP; ++i) if (i < d) a[i * ld + c] = (double)v[i];
}

// evaluate the full target at th: (lp, g).  g is only meaningful when want_grad.
__device__ __forceinline__ void eval_target(EpiCtx& C, const float (&th)[kDP], bool want_grad, float& lp,
                                            float (&g)[kDP]) {
  float out;
  tc_eval(C, th, want_grad, out, g);
  if (!want_grad) {
#pragma unroll
    for (int i = 0; i < kDP; ++i) g[i] = 0.0f;
  }
  finish_target(C, th, out, want_grad, lp, g);
}

}  // namespace tc
}  // namespace best
