// Epilogue / sampler side of the fused tensor-core kernel.  Included by tc_fused.cu only.
//
// 16 epilogue warps = 512 threads.  Thread (row, k): row = TMEM lane = chain, k = 0..3.
//   * MLP epilogues: of every 64-column group the thread handles columns [16k, 16k+16).
//   * sampler algebra: the thread owns parameter dimensions [8k, 8k+8) of its chain; the four
//     threads of a chain (same lane, four different warps of one TMEM lane quarter) exchange
//     matvec inputs and partial sums through SMEM with a 128-thread named barrier.
//   * geometries 128 / 256 (Geo::kOwn): in every N-chunk but the last of an op warp k instead OWNS the
//     64-column groups grp = k (mod 4) and walks them in four 16-column pieces (one publish per 64 columns).
// The r1a profile (profiles/r1a_hmc_ncu_full.md) showed these warps to be ISSUE-bound (62.6 k
// issue cycles per evaluation against 50.7 k MMA cycles), so everything here is written for
// instruction count: 32-bit shared-space addresses, packed f32x2 math, one MUFU per element,
// per-thread addresses hoisted into EpiCtx.
#pragma once

namespace best {
namespace tc {

using ptx::f32x2;

struct EpiCtx {
  const Params* P;
  Bars bars;
  uint32_t sbase;       // shared-space address of the carve-up base
  uint32_t tmem_lane;   // tmem base + (lane quarter << 16)
  int row;              // 0..127
  int k;                // 0..3
  uint32_t a_wr;        // ping-pong geometry: byte offset of the operand buffer this op's epilogue writes
  int to_leader;        // CTA pair, rank 1: a_ready / d_free arrivals go to the leader CTA's barriers
  int half;             // CTA pair: 0 = lanes 0..63 (lower N half, runs the sampler), 1 = lanes 64..127
  uint32_t o, g;        // op / n-chunk counters (mirror the MMA issuer)
  uint32_t vslot, pslot;  // rotating scratch slots
  uint32_t emit_pending;  // this thread has committed a bulk copy out of the row staging area (emit_tile)
  // per-thread constants
  uint32_t a_thr0, a_thr1;  // shared addresses of this thread's two 16-B pieces in A k-chunk 0 (SW128)
  uint32_t bias_thr;        // shared address of bias[0][16k]
  uint32_t wouts_thr;       // shared address of (s * w_out)[16k]
  uint32_t v_thr;           // byte offset of this row inside an exchange slot: row * 8
  uint8_t* dact_thr;        // global: this thread's 16 bytes inside act' block (layer 0, chunk 0)
  uint8_t* aimg_thr;        // L2-image tiles: global image of the next A operand, this thread's first 16-B piece
};

// arrive on a barrier the MMA issuer waits on: the CTA's own, or (second CTA of a pair) the leader's.
// One arrival per THREAD: one per warp (lane 0 after __syncwarp) was measured 1-2 % slower on B200.
__device__ __forceinline__ void arrive_mma(const EpiCtx& C, uint32_t bar) {
  if (C.to_leader) ptx::mbar_arrive_leader(bar);
  else ptx::mbar_arrive(bar);
}

// the owner of a k-chunk arrives for the row's four threads
__device__ __forceinline__ void arrive_mma4(const EpiCtx& C, uint32_t bar) {
  if (C.to_leader) ptx::mbar_arrive4_leader(bar);
  else ptx::mbar_arrive4(bar);
}

// bias of the thread's 16 columns of group jn as 8 fp32 pairs
template <int ROWS>
__device__ __forceinline__ void load_bias(const EpiCtx& C, int layer, int jn, int colofs, f32x2 (&b)[8]) {
  if (!C.P->bias16) {
    const uint32_t a = C.bias_thr + (uint32_t)(layer * C.P->H + jn * 64 + colofs) * 4u;
#pragma unroll
    for (int i = 0; i < 4; ++i) ptx::lds_c2x64(a + i * 16, b[2 * i], b[2 * i + 1]);
  } else {   // bf16 table (the fp32 one would not fit beside a 1024-wide layer's other tables)
    const uint32_t a = C.bias_thr + (uint32_t)(layer * C.P->H + jn * 64 + colofs) * 2u;
    unsigned long long q[4];
    ptx::lds_c2x64(a, q[0], q[1]);
    ptx::lds_c2x64(a + 16, q[2], q[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      uint32_t w0, w1;
      ptx::unpack2u(q[i], w0, w1);
      b[2 * i] = ptx::pack2u(w0 << 16, w0 & 0xFFFF0000u);
      b[2 * i + 1] = ptx::pack2u(w1 << 16, w1 & 0xFFFF0000u);
    }
  }
}
// the same from a formed shared address (pair fast path: per-chunk base, the groups address with immediates)
template <bool B16>
__device__ __forceinline__ void load_bias_at(uint32_t a, f32x2 (&b)[8]) {
  if (!B16) {
#pragma unroll
    for (int i = 0; i < 4; ++i) ptx::lds_c2x64(a + i * 16, b[2 * i], b[2 * i + 1]);
  } else {
    unsigned long long q[4];
    ptx::lds_c2x64(a, q[0], q[1]);
    ptx::lds_c2x64(a + 16, q[2], q[3]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      uint32_t w0, w1;
      ptx::unpack2u(q[i], w0, w1);
      b[2 * i] = ptx::pack2u(w0 << 16, w0 & 0xFFFF0000u);
      b[2 * i + 1] = ptx::pack2u(w1 << 16, w1 & 0xFFFF0000u);
    }
  }
}
// store the thread's 16 bf16 results of group jn as the next A operand (no fence / signal here)
template <int ROWS>
__device__ __forceinline__ void store_a(const EpiCtx& C, int jn, const uint32_t (&hp)[8]) {
  if (Geo<ROWS>::kInPlace) {
    const uint32_t off = jn * Geo<ROWS>::kAChunk + (Geo<ROWS>::kPingPong ? C.a_wr : 0u);
    ptx::sts_128(C.a_thr0 + off, hp[0], hp[1], hp[2], hp[3]);
    ptx::sts_128(C.a_thr1 + off, hp[4], hp[5], hp[6], hp[7]);
  } else {
    uint8_t* p0 = C.aimg_thr + (size_t)jn * Geo<ROWS>::kAChunk;
    uint8_t* p1 = reinterpret_cast<uint8_t*>(reinterpret_cast<uintptr_t>(p0) ^ (uintptr_t)16);
    ptx::stg_128(p0, hp[0], hp[1], hp[2], hp[3]);
    ptx::stg_128(p1, hp[4], hp[5], hp[6], hp[7]);
  }
}


// chunk-owner geometry: the thread's 16 bf16 results of piece p (columns [16p, 16p+16)) of k-chunk jn
template <int ROWS>
__device__ __forceinline__ void store_piece(const EpiCtx& C, int jn, int p, const uint32_t (&hp)[8]) {
  const uint32_t base = C.a_thr0 + (uint32_t)jn * Geo<ROWS>::kAChunk;   // a_thr0 = row base, a_thr1 = row & 7
  ptx::sts_128(base + (((uint32_t)(2 * p) ^ C.a_thr1) << 4), hp[0], hp[1], hp[2], hp[3]);
  ptx::sts_128(base + (((uint32_t)(2 * p + 1) ^ C.a_thr1) << 4), hp[4], hp[5], hp[6], hp[7]);
}

__device__ __forceinline__ void qbar(const EpiCtx& C) { ptx::named_bar_sync(1 + (C.row >> 5), 128); }

// The forward weights and biases of every SiLU hidden layer are packed pre-scaled by 1/2 (exact in
// bf16), so the accumulator holds a/2 and, with t = tanh(a/2),
//   sigma(a) = (1+t)/2,  h = a sigma = (a/2)(1+t),  h' = sigma + h (1 - sigma)  =>  e := 2 h' - 1 = t + h (1 - t)
// costs one MUFU and three FFMA2 per element pair.  The scratch holds e (bf16), not h': the backward weights are
// packed pre-scaled by 1/2 as well (exact), so the backward accumulator is v = (delta W)/2 and
// delta_prev = (delta W) h' = v (e + 1) = fma(v, e, v) -- one instruction, as the plain product was.
// tanh.approx has ~2^-11 relative error, below the 2^-9 of the bf16 rounding that follows.
constexpr bool kSiluHalfPrescale = true;

__device__ __forceinline__ void silu_pair(f32x2 a, f32x2& h, f32x2& e) {
  float x0, x1;
  ptx::unpack2(a, x0, x1);   // a holds (pre-activation)/2
  const f32x2 t = ptx::pack2(ptx::tanh_approx(x0), ptx::tanh_approx(x1));
  h = ptx::fma2(a, t, a);
  const f32x2 om = ptx::fma2(t, ptx::pack2(-1.0f, -1.0f), ptx::pack2(1.0f, 1.0f));
  e = ptx::fma2(h, om, t);
}
__device__ __forceinline__ void tanh_pair(f32x2 a, f32x2& h, f32x2& e) {   // h' = 1 - h^2, e = 2 h' - 1 = 1 - 2 h^2
  float x0, x1;
  ptx::unpack2(a, x0, x1);
  h = ptx::pack2(ptx::tanh_approx(x0), ptx::tanh_approx(x1));
  e = ptx::fma2(ptx::mul2(h, h), ptx::pack2(-2.0f, -2.0f), ptx::pack2(1.0f, 1.0f));
}

// ---- first A operand: theta split into bf16 hi | lo (own 8 dims -> pieces k and 4+k) ------------
template <int ROWS>
__device__ __forceinline__ void write_xin(EpiCtx& C, const float (&th)[8]) {
  if (Geo<ROWS>::kPair && C.half != 0) return;   // the upper lane half only takes part in the MLP epilogues
  if (C.emit_pending) {   // the row staging area (operand bytes 48-64 KB) is about to become operand again
    ptx::bulk_wait_read0();
    C.emit_pending = 0;
  }
  if (!Geo<ROWS>::kPingPong) ptx::mbar_wait(C.bars.a_free(0), (C.o & 1u) ^ 1u);
  uint32_t hi[4], lo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t h2 = ptx::pack_bf16x2(th[2 * i], th[2 * i + 1]);
    hi[i] = h2;
    lo[i] = ptx::pack_bf16x2(th[2 * i] - ptx::bf16_lo(h2), th[2 * i + 1] - ptx::bf16_hi(h2));
  }
  const uint32_t rowa = C.sbase + SmemLayout::A + C.row * 128;
  ptx::sts_128(rowa + (((uint32_t)C.k ^ (C.row & 7)) << 4), hi[0], hi[1], hi[2], hi[3]);
  ptx::sts_128(rowa + (((uint32_t)(4 + C.k) ^ (C.row & 7)) << 4), lo[0], lo[1], lo[2], lo[3]);
  ptx::fence_proxy_async();
  if ((!Geo<ROWS>::kInPlace)) {
    ptx::mbar_arrive(C.bars.xin_done());   // warp 3 publishes a_ready
  } else {
    for (int j = 0; j < C.P->kch_max; ++j) arrive_mma(C, C.bars.a_ready(j));
  }
}

// ---- MLP epilogues --------------------------------------------------------------------------
// The epilogue warps are latency-bound (r1 timing decomposition): per 64-column
// group a warp pays a TMEM load, an mbarrier wait, a proxy fence (MEMBAR + FENCE) and an arrive,
// each a serialised 50-200 cycle stall.  The next op's MMAs wait on exactly these signals, so the
// operand is published per 64-column group (publishing 128 columns at a time with one fence was
// measured 10 % SLOWER); the a_free wait is skipped in the last N-chunk (its d_full commit is
// ordered after every a_free commit of the op).

// the register arithmetic of 16 columns: hp = next operand (bf16 pairs), dp = e = 2 act' - 1 (hidden layers)
template <int ACT, bool LAST>
__device__ __forceinline__ void fwd_math(const uint32_t (&v)[16], const f32x2 (&b)[8], const f32x2 (&ws)[8], bool want_grad,
                                         f32x2& acc2, uint32_t (&hp)[8], uint32_t (&dp)[8]) {
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const f32x2 a = ptx::add2(ptx::pack2u(v[2 * i], v[2 * i + 1]), b[i]);
    f32x2 h, dd;
    if (ACT == BEST_ACT_SILU) silu_pair(a, h, dd); else tanh_pair(a, h, dd);
    if (LAST) {   // ws = (s w_out)/2: the output dot product is doubled once at the end, delta = h' s w_out = (e + 1) ws
      acc2 = ptx::fma2(h, ws[i], acc2);
      if (want_grad) hp[i] = ptx::pack_bf16x2_from(ptx::fma2(dd, ws[i], ws[i]));
    } else {
      hp[i] = ptx::pack_bf16x2_from(h);
      dp[i] = ptx::pack_bf16x2_from(dd);
    }
  }
}

// bias + activation (+ act' to scratch, or delta for the last layer) of one group, in registers
template <int ACT, bool LAST, int ROWS>
__device__ __forceinline__ void fwd_group(const EpiCtx& C, int layer, int jn, int colofs, const uint32_t (&v)[16],
                                          bool want_grad, uint8_t* dact_l, f32x2& acc2, uint32_t (&hp)[8]) {
  // colofs: first column of the thread's 16 inside the 64-column group when the per-thread bases do not hold
  // it already (chunk-owner geometry: 16 p; otherwise 0)
  constexpr uint32_t kDBlk = Geo<ROWS>::kTileRows * 128, kDPiece = Geo<ROWS>::kTileRows * 16;
  f32x2 b[8];
  load_bias<ROWS>(C, layer, jn, colofs, b);
  f32x2 ws[8];
  if (LAST) {
#pragma unroll
    for (int i = 0; i < 4; ++i) ptx::lds_c2x64(C.wouts_thr + jn * 256 + colofs * 4 + i * 16, ws[2 * i], ws[2 * i + 1]);
  }
  uint32_t dp[8];
  fwd_math<ACT, LAST>(v, b, ws, want_grad, acc2, hp, dp);
  if (!LAST && want_grad) {
    uint8_t* dptr = dact_l + (size_t)jn * kDBlk + (size_t)(colofs >> 3) * kDPiece;
    ptx::stg_128(dptr, dp[0], dp[1], dp[2], dp[3]);
    ptx::stg_128(dptr + kDPiece, dp[4], dp[5], dp[6], dp[7]);
  }
}

// publish groups jn0 .. jn0+n-1 of the next operand (stores already issued)
template <int ROWS>
__device__ __forceinline__ void publish_a(EpiCtx& C, int jn0, int n) {
  if (Geo<ROWS>::kInPlace) {
    ptx::fence_proxy_async();
    for (int i = 0; i < n; ++i) arrive_mma(C, C.bars.a_ready(jn0 + i));
  }
}

// CTA pair: the 64-column block of the layer that lane half `half` finds in its group `grp` of N-chunk c.
// The hardware puts N columns [128 half, +128) of the chunk in that half's lanes; paired ops are packed
// with the chunk's four 64-row blocks of B in the order 0,2,1,3, so that one round of the epilogue (both
// halves, same grp) completes two CONSECUTIVE k-chunks of the next operand.
__device__ __forceinline__ int pair_jn(const OpDesc& op, int c, int half, int grp, int ngrp) {
  return op.perm ? c * (op.ncols >> 6) + grp * 2 + half : c * (op.ncols >> 6) + half * ngrp + grp;
}

// forward epilogue of one op
template <int ACT, bool LAST, int ROWS>
__device__ __forceinline__ void epi_fwd(EpiCtx& C, const OpDesc& op, bool want_grad, f32x2& acc2,
                                        int& written) {
  const bool writes_a = !(LAST && !want_grad);
  // 64-column groups of this thread per N-chunk (CTA pair: the lane half owns half of the chunk)
  const int ngrp = Geo<ROWS>::kPair ? (op.ncols >> 7) : (op.ncols >> 6);
  constexpr uint32_t kDBlk = Geo<ROWS>::kTileRows * 128;
  uint8_t* dact_l = C.dact_thr + (size_t)(op.layer * (C.P->H >> 6)) * kDBlk;
  for (int c = 0; c < op.nch; ++c, ++C.g) {
    const uint32_t buf = C.g % Geo<ROWS>::kNBuf, use = C.g / Geo<ROWS>::kNBuf;
    ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
    ptx::tc_fence_after();
    const uint32_t tcol = C.tmem_lane + buf * Geo<ROWS>::kBufCols + C.k * 16;
    const bool gate = Geo<ROWS>::kInPlace && !Geo<ROWS>::kPingPong && writes_a && (c != op.nch - 1);
    if (Geo<ROWS>::kOwn) {
      const uint32_t tbase = C.tmem_lane + buf * Geo<ROWS>::kBufCols;
      if (!Geo<ROWS>::kOwnLastInterleaved || c != op.nch - 1 || !writes_a) {   // owner order
        for (int grp = C.k; grp < ngrp; grp += 4) {
          const int jn = c * ngrp + grp;
          // per-group bases once, the four pieces address with immediates (the owner geometries keep the fp32 bias table)
          constexpr uint32_t kDBlk = Geo<ROWS>::kTileRows * 128, kDPiece = Geo<ROWS>::kTileRows * 16;
          const uint32_t bias_a = C.bias_thr + (uint32_t)(op.layer * C.P->H + jn * 64) * 4u;
          const uint32_t ws_a = C.wouts_thr + (uint32_t)jn * 256u;
          const uint32_t sts_a = C.a_thr0 + (uint32_t)jn * Geo<ROWS>::kAChunk, x7 = C.a_thr1 << 4;
          uint8_t* dact_a = dact_l + (size_t)jn * kDBlk;
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            uint32_t v[16], hp[8], dp[8];
            ptx::tmem_ld16(tbase + grp * 64 + p * 16, v);
            f32x2 b[8], ws[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) ptx::lds_c2x64(bias_a + p * 64 + i * 16, b[2 * i], b[2 * i + 1]);
            if (LAST) {
#pragma unroll
              for (int i = 0; i < 4; ++i) ptx::lds_c2x64(ws_a + p * 64 + i * 16, ws[2 * i], ws[2 * i + 1]);
            }
            ptx::tmem_ld_wait();
            fwd_math<ACT, LAST>(v, b, ws, want_grad, acc2, hp, dp);
            if (!LAST && want_grad) {
              ptx::stg_128(dact_a + (2 * p) * kDPiece, dp[0], dp[1], dp[2], dp[3]);
              ptx::stg_128(dact_a + (2 * p + 1) * kDPiece, dp[4], dp[5], dp[6], dp[7]);
            }
            if (writes_a) {
              if (gate && p == 0) ptx::mbar_wait(C.bars.a_free(jn), C.o & 1u);
              ptx::sts_128(sts_a + ((uint32_t)(32 * p) ^ x7), hp[0], hp[1], hp[2], hp[3]);
              ptx::sts_128(sts_a + ((uint32_t)(32 * p + 16) ^ x7), hp[4], hp[5], hp[6], hp[7]);
            }
          }
          if (writes_a) {
            ptx::fence_proxy_async();
            arrive_mma4(C, C.bars.a_ready(jn));
          }
        }
      } else {   // last N-chunk: the next op's MMAs consume k-chunk after k-chunk as they are published
        // (per-chunk bases once, immediates per group; requesting the NEXT group's accumulator columns before this
        // group's arithmetic needs a second 16-register array: 4.7 KB of spills, not kept)
        constexpr uint32_t kDBlk = Geo<ROWS>::kTileRows * 128, kDPiece = Geo<ROWS>::kTileRows * 16;
        const int jn0 = c * ngrp;
        const uint32_t bias_a = C.bias_thr + (uint32_t)(op.layer * C.P->H + jn0 * 64 + 16 * C.k) * 4u;
        const uint32_t ws_a = C.wouts_thr + (uint32_t)jn0 * 256u + (uint32_t)C.k * 64u;
        const uint32_t x7 = C.a_thr1 << 4, a0 = C.a_thr0 + (uint32_t)jn0 * Geo<ROWS>::kAChunk;
        const uint32_t sts0 = a0 + ((uint32_t)(32 * C.k) ^ x7), sts1 = a0 + ((uint32_t)(32 * C.k + 16) ^ x7);
        uint8_t* dact_a = dact_l + (size_t)jn0 * kDBlk + (size_t)(2 * C.k) * kDPiece;
#pragma unroll
        for (int g0 = 0; g0 < 4; ++g0) {
          if (g0 < ngrp) {
            uint32_t v[16], hp[8], dp[8];
            f32x2 b[8], ws[8];
            ptx::tmem_ld16(tbase + g0 * 64 + C.k * 16, v);
#pragma unroll
            for (int i = 0; i < 4; ++i) ptx::lds_c2x64(bias_a + g0 * 256 + i * 16, b[2 * i], b[2 * i + 1]);
            if (LAST) {
#pragma unroll
              for (int i = 0; i < 4; ++i) ptx::lds_c2x64(ws_a + g0 * 256 + i * 16, ws[2 * i], ws[2 * i + 1]);
            }
            ptx::tmem_ld_wait();
            fwd_math<ACT, LAST>(v, b, ws, want_grad, acc2, hp, dp);
            if (!LAST && want_grad) {
              ptx::stg_128(dact_a + (size_t)g0 * kDBlk, dp[0], dp[1], dp[2], dp[3]);
              ptx::stg_128(dact_a + (size_t)g0 * kDBlk + kDPiece, dp[4], dp[5], dp[6], dp[7]);
            }
            ptx::sts_128(sts0 + g0 * Geo<ROWS>::kAChunk, hp[0], hp[1], hp[2], hp[3]);
            ptx::sts_128(sts1 + g0 * Geo<ROWS>::kAChunk, hp[4], hp[5], hp[6], hp[7]);
            ptx::fence_proxy_async();
            arrive_mma(C, C.bars.a_ready(jn0 + g0));
          }
        }
      }
      ptx::tc_fence_before();
      arrive_mma(C, C.bars.d_free(buf));
      continue;
    }
    if (Geo<ROWS>::kPair && op.perm && ngrp == 2) {
      // CTA pairs, permuted row blocks, N = 256: this lane half's two groups are the k-chunks jn0 and jn0 + 2 of the
      // next operand.  Per-chunk bases once, the groups address with immediates; bias (and output row) requested
      // under the TMEM load (as in the owner geometries; same arithmetic as the general loop below, same bits)
      constexpr uint32_t kDPiece = Geo<ROWS>::kTileRows * 16;
      const int jn0 = c * 4 + C.half;
      const bool b16 = C.P->bias16 != 0;
      const uint32_t bias_a = C.bias_thr + (uint32_t)(op.layer * C.P->H + jn0 * 64) * (b16 ? 2u : 4u);
      const uint32_t ws_a = C.wouts_thr + (uint32_t)jn0 * 256u;
      const uint32_t aoff = (uint32_t)jn0 * Geo<ROWS>::kAChunk + (Geo<ROWS>::kPingPong ? C.a_wr : 0u);
      const uint32_t sts0 = C.a_thr0 + aoff, sts1 = C.a_thr1 + aoff;
      uint8_t* dact_a = dact_l + (size_t)jn0 * kDBlk;
      const uint32_t bar_r = C.bars.a_ready(jn0), bar_f = C.bars.a_free(jn0);
#pragma unroll
      for (int g0 = 0; g0 < 2; ++g0) {
        uint32_t v[16], hp[8], dp[8];
        f32x2 b[8], ws[8];
        ptx::tmem_ld16(tcol + g0 * 64, v);
        if (b16) load_bias_at<true>(bias_a + g0 * 256, b); else load_bias_at<false>(bias_a + g0 * 512, b);
        if (LAST) {
#pragma unroll
          for (int i = 0; i < 4; ++i) ptx::lds_c2x64(ws_a + g0 * 512 + i * 16, ws[2 * i], ws[2 * i + 1]);
        }
        ptx::tmem_ld_wait();
        fwd_math<ACT, LAST>(v, b, ws, want_grad, acc2, hp, dp);
        if (!LAST && want_grad) {
          ptx::stg_128(dact_a + (size_t)(2 * g0) * kDBlk, dp[0], dp[1], dp[2], dp[3]);
          ptx::stg_128(dact_a + (size_t)(2 * g0) * kDBlk + kDPiece, dp[4], dp[5], dp[6], dp[7]);
        }
        if (writes_a) {
          if (gate) ptx::mbar_wait(bar_f + g0 * 16, C.o & 1u);
          ptx::sts_128(sts0 + g0 * 2 * Geo<ROWS>::kAChunk, hp[0], hp[1], hp[2], hp[3]);
          ptx::sts_128(sts1 + g0 * 2 * Geo<ROWS>::kAChunk, hp[4], hp[5], hp[6], hp[7]);
          ptx::fence_proxy_async();
          arrive_mma(C, bar_r + g0 * 16);
        }
      }
      if (writes_a) written = max(written, jn0 + 3);
    } else
    for (int g0 = 0; g0 < ngrp; ++g0) {
      const int grp = g0;
      const int jn = Geo<ROWS>::kPair ? pair_jn(op, c, C.half, grp, ngrp) : c * ngrp + grp;
      uint32_t v[16], hp[8];
      ptx::tmem_ld16(tcol + grp * 64, v);
      ptx::tmem_ld_wait();
      fwd_group<ACT, LAST, ROWS>(C, op.layer, jn, 0, v, want_grad, dact_l, acc2, hp);
      if (writes_a) {
        if (gate) ptx::mbar_wait(C.bars.a_free(jn), C.o & 1u);
        store_a<ROWS>(C, jn, hp);
        publish_a<ROWS>(C, jn, 1);
        written = max(written, jn + 1);
      }
    }
    if ((!Geo<ROWS>::kInPlace) && writes_a) {   // this N-chunk of the next operand is in the L2 image
      ptx::fence_proxy_async_all();
      ptx::mbar_arrive(C.bars.epi_done(c));
    }
    ptx::tc_fence_before();
    arrive_mma(C, C.bars.d_free(buf));
  }
  if (Geo<ROWS>::kOwn && writes_a) written = op.nch * ngrp;   // (all k-chunks, by their owners)
}

// backward epilogue: delta_{l-1} = (delta_l W_l) .* act'_{l-1}
template <int ROWS>
__device__ __forceinline__ void bwd_group(const uint32_t (&v)[16], const uint4& d0, const uint4& d1,
                                          uint32_t (&hp)[8]) {
  const uint32_t dw[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const f32x2 dd = ptx::pack2u(dw[i] << 16, dw[i] & 0xFFFF0000u);
    const f32x2 vv = ptx::pack2u(v[2 * i], v[2 * i + 1]);   // (delta W)/2; dd holds e = 2 act' - 1
    hp[i] = ptx::pack_bf16x2_from(ptx::fma2(vv, dd, vv));
  }
}
template <int ROWS>
__device__ __forceinline__ void epi_bwd(EpiCtx& C, const OpDesc& op, int& written) {
  // 64-column groups of this thread per N-chunk (CTA pair: the lane half owns half of the chunk)
  const int ngrp = Geo<ROWS>::kPair ? (op.ncols >> 7) : (op.ncols >> 6);
  constexpr uint32_t kDBlk = Geo<ROWS>::kTileRows * 128, kDPiece = Geo<ROWS>::kTileRows * 16;
  const uint8_t* dact_l = C.dact_thr + (size_t)(op.layer * (C.P->H >> 6)) * kDBlk;
  const int jstep = (Geo<ROWS>::kPair && op.perm) ? 2 : 1;
  // act' is fetched one group ahead, ACROSS N-chunk boundaries as well: the first group of an op is requested
  // before its accumulator is complete, the first group of the next N-chunk while the last group of this one is
  // processed (requesting it only at the top of the chunk exposed an L2 round trip per chunk: in the N-chunk-outer
  // order the next chunk's accumulator is usually complete by then).
  if (Geo<ROWS>::kOwn) {
    // every N-chunk but the last in owner order (pieces (grp = k mod 4, p = 0..3)), the last one interleaved (all
    // four threads of a row on group g0, columns [16k, 16k+16)); act' of the NEXT piece is requested while the
    // current one is processed, across group and N-chunk boundaries as well
    const int last = op.nch - 1;
    auto owner_chunk = [&](int c) -> bool { return !Geo<ROWS>::kOwnLastInterleaved || c != last; };
    auto piece_ptr = [&](int c, int i) -> const uint8_t* {   // i-th piece of this thread in N-chunk c (ngrp <= 4)
      return owner_chunk(c) ? dact_l + (size_t)(c * ngrp + C.k) * kDBlk + (size_t)(2 * i) * kDPiece
                            : dact_l + (size_t)(c * ngrp + i) * kDBlk + (size_t)(2 * C.k) * kDPiece;
    };
    uint4 a0 = make_uint4(0, 0, 0, 0), a1 = a0;
    if (!owner_chunk(0) || C.k < ngrp) {   // (an op has one or two N-chunks; with two, ngrp = 4 > k)
      const uint8_t* dp = piece_ptr(0, 0);
      a0 = ptx::ldg_128(dp); a1 = ptx::ldg_128(dp + kDPiece);
    }
    for (int c = 0; c < op.nch; ++c, ++C.g) {
      const uint32_t buf = C.g % Geo<ROWS>::kNBuf, use = C.g / Geo<ROWS>::kNBuf;
      ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
      ptx::tc_fence_after();
      const uint32_t tbase = C.tmem_lane + buf * Geo<ROWS>::kBufCols;
      const uint32_t x7 = C.a_thr1 << 4;
      if (!Geo<ROWS>::kOwnLastInterleaved || c != last) {   // owner order
        const int jn = c * ngrp + C.k;
        if (C.k < ngrp) {
          // bases once per group, immediates per piece (as in epi_fwd)
          const uint8_t* dact_a = dact_l + (size_t)jn * kDBlk;
          const uint8_t* dact_n = (c + 1 < op.nch) ? piece_ptr(c + 1, 0) : dact_a;   // first piece of the next N-chunk
          const uint32_t sts_a = C.a_thr0 + (uint32_t)jn * Geo<ROWS>::kAChunk;
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            uint32_t v[16], hp[8];
            ptx::tmem_ld16(tbase + C.k * 64 + p * 16, v);
            const uint4 d0 = a0, d1 = a1;
            if (p < 3) {
              a0 = ptx::ldg_128(dact_a + (2 * p + 2) * kDPiece); a1 = ptx::ldg_128(dact_a + (2 * p + 3) * kDPiece);
            } else if (c + 1 < op.nch) {
              a0 = ptx::ldg_128(dact_n); a1 = ptx::ldg_128(dact_n + kDPiece);
            }
            ptx::tmem_ld_wait();
            bwd_group<ROWS>(v, d0, d1, hp);
            if (p == 0) ptx::mbar_wait(C.bars.a_free(jn), C.o & 1u);
            ptx::sts_128(sts_a + ((uint32_t)(32 * p) ^ x7), hp[0], hp[1], hp[2], hp[3]);
            ptx::sts_128(sts_a + ((uint32_t)(32 * p + 16) ^ x7), hp[4], hp[5], hp[6], hp[7]);
          }
          ptx::fence_proxy_async();
          arrive_mma4(C, C.bars.a_ready(jn));
        }
      } else {
        const int jn0 = c * ngrp;
        const uint8_t* dact_a = dact_l + (size_t)jn0 * kDBlk + (size_t)(2 * C.k) * kDPiece;   // + g0 * kDBlk
        const uint32_t a0s = C.a_thr0 + (uint32_t)jn0 * Geo<ROWS>::kAChunk;
        const uint32_t sts0 = a0s + ((uint32_t)(32 * C.k) ^ x7), sts1 = a0s + ((uint32_t)(32 * C.k + 16) ^ x7);
#pragma unroll
        for (int g0 = 0; g0 < 4; ++g0) {
          if (g0 < ngrp) {
            uint32_t v[16], hp[8];
            ptx::tmem_ld16(tbase + g0 * 64 + C.k * 16, v);
            const uint4 d0 = a0, d1 = a1;
            if (g0 + 1 < ngrp) {
              a0 = ptx::ldg_128(dact_a + (size_t)(g0 + 1) * kDBlk); a1 = ptx::ldg_128(dact_a + (size_t)(g0 + 1) * kDBlk + kDPiece);
            }
            ptx::tmem_ld_wait();
            bwd_group<ROWS>(v, d0, d1, hp);
            ptx::sts_128(sts0 + g0 * Geo<ROWS>::kAChunk, hp[0], hp[1], hp[2], hp[3]);
            ptx::sts_128(sts1 + g0 * Geo<ROWS>::kAChunk, hp[4], hp[5], hp[6], hp[7]);
            ptx::fence_proxy_async();
            arrive_mma(C, C.bars.a_ready(jn0 + g0));
          }
        }
      }
      ptx::tc_fence_before();
      arrive_mma(C, C.bars.d_free(buf));
    }
    written = op.nch * ngrp;
    return;
  }
  uint4 a0, a1;
  {
    const int jnc0 = Geo<ROWS>::kPair ? pair_jn(op, 0, C.half, 0, ngrp) : 0;
    const uint8_t* dp = dact_l + (size_t)jnc0 * kDBlk;
    a0 = ptx::ldg_128(dp); a1 = ptx::ldg_128(dp + kDPiece);
  }
  for (int c = 0; c < op.nch; ++c, ++C.g) {
    const uint32_t buf = C.g % Geo<ROWS>::kNBuf, use = C.g / Geo<ROWS>::kNBuf;
    const bool gate = Geo<ROWS>::kInPlace && !Geo<ROWS>::kPingPong && (c != op.nch - 1);
    const int jnc = Geo<ROWS>::kPair ? pair_jn(op, c, C.half, 0, ngrp) : c * ngrp;   // group 0 of this chunk
    const int jnc_next = Geo<ROWS>::kPair ? pair_jn(op, c + 1, C.half, 0, ngrp) : (c + 1) * ngrp;
    ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
    ptx::tc_fence_after();
    const uint32_t tcol = C.tmem_lane + buf * Geo<ROWS>::kBufCols + C.k * 16;
    if (Geo<ROWS>::kPair && op.perm && ngrp == 2) {
      // (see epi_fwd) k-chunks jnc and jnc + 2; act' of the next group / of the next N-chunk's first group (jnc + 4)
      // is requested under the TMEM load
      const uint8_t* dact_a = dact_l + (size_t)jnc * kDBlk;
      const uint32_t aoff = (uint32_t)jnc * Geo<ROWS>::kAChunk + (Geo<ROWS>::kPingPong ? C.a_wr : 0u);
      const uint32_t sts0 = C.a_thr0 + aoff, sts1 = C.a_thr1 + aoff;
      const uint32_t bar_r = C.bars.a_ready(jnc), bar_f = C.bars.a_free(jnc);
      const bool more = c + 1 < op.nch;
#pragma unroll
      for (int g0 = 0; g0 < 2; ++g0) {
        uint32_t v[16], hp[8];
        ptx::tmem_ld16(tcol + g0 * 64, v);
        const uint4 d0 = a0, d1 = a1;
        if (g0 == 0 || more) {
          a0 = ptx::ldg_128(dact_a + (size_t)(2 * g0 + 2) * kDBlk); a1 = ptx::ldg_128(dact_a + (size_t)(2 * g0 + 2) * kDBlk + kDPiece);
        }
        ptx::tmem_ld_wait();
        bwd_group<ROWS>(v, d0, d1, hp);
        if (gate) ptx::mbar_wait(bar_f + g0 * 16, C.o & 1u);
        ptx::sts_128(sts0 + g0 * 2 * Geo<ROWS>::kAChunk, hp[0], hp[1], hp[2], hp[3]);
        ptx::sts_128(sts1 + g0 * 2 * Geo<ROWS>::kAChunk, hp[4], hp[5], hp[6], hp[7]);
        ptx::fence_proxy_async();
        arrive_mma(C, bar_r + g0 * 16);
      }
      written = max(written, jnc + 3);
    } else
    for (int g0 = 0; g0 < ngrp; ++g0) {
      const int grp = g0;
      const int jn = jnc + grp * jstep;
      uint32_t v[16], hp[8];
      ptx::tmem_ld16(tcol + grp * 64, v);
      const uint4 d0 = a0, d1 = a1;
      if (g0 + 1 < ngrp || c + 1 < op.nch) {   // prefetch the next group's act'
        const int jnn = (g0 + 1 < ngrp) ? jnc + (g0 + 1) * jstep
                                        : jnc_next;
        const uint8_t* dn = dact_l + (size_t)jnn * kDBlk;
        a0 = ptx::ldg_128(dn); a1 = ptx::ldg_128(dn + kDPiece);
      }
      ptx::tmem_ld_wait();
      bwd_group<ROWS>(v, d0, d1, hp);
      if (gate) ptx::mbar_wait(C.bars.a_free(jn), C.o & 1u);
      store_a<ROWS>(C, jn, hp);
      publish_a<ROWS>(C, jn, 1);
      written = max(written, jn + 1);
    }
    if (!Geo<ROWS>::kInPlace) {
      ptx::fence_proxy_async_all();
      ptx::mbar_arrive(C.bars.epi_done(c));
    }
    ptx::tc_fence_before();
    arrive_mma(C, C.bars.d_free(buf));
  }
}



// One MLP evaluation.  In: own 8 dims of theta.  Out: this thread's PARTIAL of s * MLP output
// (over its columns, without the output bias) and, when want_grad, s * d MLP / d theta for its
// own 8 dims.
template <int ROWS>
__device__ __forceinline__ void tc_eval(EpiCtx& C, const float (&th)[8], bool want_grad, float& out_part,
                                        float (&gm)[8]) {
  const Params& P = *C.P;
  write_xin<ROWS>(C, th);
  f32x2 acc2 = ptx::pack2(0.0f, 0.0f);
  const int n_ops = want_grad ? P.n_ops_all : P.n_ops_fwd;
  for (int oi = 0; oi < n_ops; ++oi, ++C.o) {
    const OpDesc op = P.ops[oi];
    int written = 0;
    C.a_wr = (uint32_t)((oi + 1) & 1) * (uint32_t)Geo<ROWS>::kPPStride;   // (ping-pong) the buffer the NEXT op reads
    if (op.epi == EPI_FWD_HID) {
      if (P.act == BEST_ACT_SILU) epi_fwd<BEST_ACT_SILU, false, ROWS>(C, op, want_grad, acc2, written);
      else epi_fwd<BEST_ACT_TANH, false, ROWS>(C, op, want_grad, acc2, written);
    } else if (op.epi == EPI_FWD_LAST) {
      if (P.act == BEST_ACT_SILU) epi_fwd<BEST_ACT_SILU, true, ROWS>(C, op, want_grad, acc2, written);
      else epi_fwd<BEST_ACT_TANH, true, ROWS>(C, op, want_grad, acc2, written);
    } else if (op.epi == EPI_BWD_HID) {
      epi_bwd<ROWS>(C, op, written);
    } else {  // EPI_BWD_FINAL: D[128][32] -> own 8 columns
      const uint32_t buf = C.g % Geo<ROWS>::kNBuf, use = C.g / Geo<ROWS>::kNBuf;
      ptx::mbar_wait(C.bars.d_full(buf), use & 1u);
      ptx::tc_fence_after();
      if (!Geo<ROWS>::kPair) {
        uint32_t v[8];
        ptx::tmem_ld8(C.tmem_lane + buf * Geo<ROWS>::kBufCols + C.k * 8, v);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 8; ++i) gm[i] = __uint_as_float(v[i]);
      } else {
        // pair layout: lanes 0..63 hold gradient dims 0..15, lanes 64..127 dims 16..31 (TMEM columns
        // 0..15 each); the k == 0 thread of each lane half hands them to the chain's sampler threads
        // through SMEM [32 dims][64 rows] (chunk 6 of the operand buffer: every MMA has completed)
        const uint32_t GX = C.sbase + SmemLayout::A + 49152u + (uint32_t)C.row * 4u;
        if (C.k == 0) {
          uint32_t v[16];
          ptx::tmem_ld16(C.tmem_lane + buf * Geo<ROWS>::kBufCols, v);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 16; ++i) ptx::sts_32(GX + (uint32_t)(C.half * 16 + i) * 256u, __uint_as_float(v[i]));
        }
        ptx::named_bar_sync(5 + (C.row >> 5), 256);
        if (C.half == 0) {
#pragma unroll
          for (int i = 0; i < 8; ++i) gm[i] = ptx::lds_32(GX + (uint32_t)(8 * C.k + i) * 256u);
        }
      }
      ptx::tc_fence_before();
      arrive_mma(C, C.bars.d_free(buf));
      ++C.g;
    }
    if ((!Geo<ROWS>::kInPlace)) {   // keep every epi_done barrier at one phase per op (written = 64-column groups)
      for (int c = (written * 64 + op.ncols - 1) / op.ncols; c < 4; ++c) ptx::mbar_arrive(C.bars.epi_done(c));
    } else if (oi != n_ops - 1) {  // keep every a_ready barrier at one phase per op
      if (!Geo<ROWS>::kPair) {
        for (int j = written; j < C.P->kch_max; ++j) arrive_mma(C, C.bars.a_ready(j));
      } else if (written == 0 && C.half == 0) {   // pair: an op writes all k-chunks or none
        for (int j = 0; j < C.P->kch_max; ++j) arrive_mma(C, C.bars.a_ready(j));
      }
    }
  }
  float a0, a1;
  ptx::unpack2(acc2, a0, a1);
  out_part = 2.0f * (a0 + a1);   // (the table holds (s w_out)/2)
  if (Geo<ROWS>::kPair) {   // the output dot product is split over both lane halves
    const uint32_t PX = C.sbase + SmemLayout::PART + 1024u + (uint32_t)C.row * 16u + (uint32_t)C.k * 4u;
    if (C.half == 1) ptx::sts_32(PX, out_part);
    ptx::named_bar_sync(5 + (C.row >> 5), 256);
    if (C.half == 0) out_part += ptx::lds_32(PX);
    ptx::named_bar_sync(5 + (C.row >> 5), 256);   // PX may be rewritten by the next evaluation
  }
}

// ---- cooperative per-chain algebra: each thread owns dims [8k, 8k+8) ---------------------------
// Exchange slot layout: [16 dim pairs][128 rows][2] floats (16 KB, rotating between A chunks 1 and
// 2, which are idle between evaluations): a thread publishes its 8 values with four STS.64 and
// reads any pair of dims of its own chain with one LDS.64.
__device__ __forceinline__ uint32_t share(EpiCtx& C, const float (&x)[8]) {
  C.vslot ^= 1u;
  const uint32_t V = C.sbase + SmemLayout::A + (1 + C.vslot) * kAChunkBytes + C.v_thr;
#pragma unroll
  for (int m = 0; m < 4; ++m) ptx::sts_64(V + (uint32_t)(4 * C.k + m) * 1024u, ptx::pack2(x[2 * m], x[2 * m + 1]));
  qbar(C);
  return V;
}
// out[i] = sum_{j in [j0, j1)} M[j][8k + i] * x_j   (j0, j1 even; M is a [32][32] float table)
__device__ __forceinline__ void mv_rows(const EpiCtx& C, uint32_t M, uint32_t V, int j0, int j1,
                                        float (&out)[8]) {
  f32x2 o[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) o[i] = ptx::pack2(0.0f, 0.0f);
  const uint32_t Mk = M + (uint32_t)C.k * 32u;
  for (int jp = j0 >> 1; jp < (j1 >> 1); ++jp) {
    float v0, v1;
    ptx::unpack2(ptx::lds_64(V + (uint32_t)jp * 1024u), v0, v1);
    f32x2 m0, m1, m2, m3;
    ptx::lds_c2x64(Mk + (uint32_t)jp * 256u, m0, m1);
    ptx::lds_c2x64(Mk + (uint32_t)jp * 256u + 16u, m2, m3);
    const f32x2 vv0 = ptx::pack2(v0, v0);
    o[0] = ptx::fma2(m0, vv0, o[0]); o[1] = ptx::fma2(m1, vv0, o[1]);
    o[2] = ptx::fma2(m2, vv0, o[2]); o[3] = ptx::fma2(m3, vv0, o[3]);
    ptx::lds_c2x64(Mk + (uint32_t)jp * 256u + 128u, m0, m1);
    ptx::lds_c2x64(Mk + (uint32_t)jp * 256u + 144u, m2, m3);
    const f32x2 vv1 = ptx::pack2(v1, v1);
    o[0] = ptx::fma2(m0, vv1, o[0]); o[1] = ptx::fma2(m1, vv1, o[1]);
    o[2] = ptx::fma2(m2, vv1, o[2]); o[3] = ptx::fma2(m3, vv1, o[3]);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) ptx::unpack2(o[i], out[2 * i], out[2 * i + 1]);
}
// out = L x : out_i = sum_{j<=i} L[i][j] x_j, own i  -> coefficients LT[j][i], j in [0, 8k+8)
__device__ __forceinline__ void mv_L(EpiCtx& C, const float (&x)[8], float (&out)[8]) {
  const uint32_t V = share(C, x);
  mv_rows(C, C.sbase + SmemLayout::LTMAT, V, 0, 8 * C.k + 8, out);
}
// out = L^T x : out_j = sum_{i>=j} L[i][j] x_i, own j -> coefficients L[i][j], i in [8k, 32)
__device__ __forceinline__ void mv_Lt(EpiCtx& C, const float (&x)[8], float (&out)[8]) {
  const uint32_t V = share(C, x);
  mv_rows(C, C.sbase + SmemLayout::LMAT, V, 8 * C.k, kDP, out);
}
// sum of one value per thread over the four threads of a chain (same result on all four)
__device__ __forceinline__ float reduce4(EpiCtx& C, float x) {
  C.pslot ^= 1u;
  const uint32_t Pp = C.sbase + SmemLayout::PART + C.pslot * 2048u + (uint32_t)C.row * 16u;
  ptx::sts_32(Pp + (uint32_t)C.k * 4u, x);
  qbar(C);
  const float4 p = ptx::lds_128f(Pp);
  return (p.x + p.y) + (p.z + p.w);
}

// full target from the MLP partial output + Gaussian (y = R r), banana and box terms.
// lp is identical on the four threads of a chain; g covers the thread's own 8 dims.
__device__ __forceinline__ void finish_target(EpiCtx& C, const float (&th)[8], float out_part, bool want_grad,
                                              float& lp, float (&g)[8]) {
  const Params& P = *C.P;
  const uint32_t vecs = C.sbase + SmemLayout::VECS;
  float part = out_part;
  float ti = 0.0f, tj = 0.0f;
  if (P.has_gauss || P.banana_i >= 0) {
    float r[8], y[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) r[i] = th[i] - ptx::lds_c32(vecs + (uint32_t)(8 * C.k + i) * 4u);
    const uint32_t V = share(C, r);
    if (P.banana_i >= 0) {
      ti = ptx::lds_32(V + (uint32_t)(P.banana_i >> 1) * 1024u + (uint32_t)(P.banana_i & 1) * 4u) +
           ptx::lds_c32(vecs + (uint32_t)P.banana_i * 4u);
      tj = ptx::lds_32(V + (uint32_t)(P.banana_j >> 1) * 1024u + (uint32_t)(P.banana_j & 1) * 4u) +
           ptx::lds_c32(vecs + (uint32_t)P.banana_j * 4u);
    }
    if (P.has_gauss) {
      mv_rows(C, C.sbase + SmemLayout::RTMAT, V, 8 * C.k, kDP, y);   // y_i = sum_{j>=i} R[i][j] r_j
#pragma unroll
      for (int i = 0; i < 8; ++i) part = fmaf(-0.5f * y[i], y[i], part);
      if (want_grad) {
        float gg[8];
        const uint32_t Vy = share(C, y);
        mv_rows(C, C.sbase + SmemLayout::RMAT, Vy, 0, 8 * C.k + 8, gg);  // (R^T y)_j = sum_{i<=j} R[i][j] y_i
#pragma unroll
        for (int i = 0; i < 8; ++i) g[i] -= gg[i];
      }
    }
  }
  if (P.has_box) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const uint32_t gi = (uint32_t)(8 * C.k + i) * 4u;
      const float lo = ptx::lds_c32(vecs + 128u + gi), hi = ptx::lds_c32(vecs + 256u + gi);
      const float ex = fmaxf(fmaxf(lo - th[i], th[i] - hi), 0.0f);
      if (ex > 0.0f && P.hard_box) {
        part = -INFINITY;   // 8(f)#1: outside the hard box
      } else if (ex > 0.0f) {
        const float iw = ptx::lds_c32(vecs + 384u + gi);
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
template <int ROWS>
__device__ __forceinline__ void eval_target(EpiCtx& C, const float (&th)[8], bool want_grad, float& lp,
                                            float (&g)[8]) {
  float out_part;
#pragma unroll
  for (int i = 0; i < 8; ++i) g[i] = 0.0f;
  tc_eval<ROWS>(C, th, want_grad, out_part, g);
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
