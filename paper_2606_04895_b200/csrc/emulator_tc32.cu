// fp32-ACCURATE emulator GEMMs on the tensor cores (north_star "bf16/fp32 variants"; "the
// fp32-accurate tensor variant (3xTF32 or bf16x3 split) ... decide by measurement").
//
// The exact path (BEST_PREC_FP32) keeps its structure -- layer-by-layer GEMMs over fp32 activations in
// L2-resident scratch, fp64 chain state, per-chain fp64 step kernels -- but for hidden widths >= 256 every GEMM
// C = epi(A B) runs as tcgen05 MMAs on SPLIT operands: a = a1 + a2 with a1 = fp16(a), a2 = fp16(a - a1) (2 x 11
// significant bits), likewise the weights, and
//     A B  ~=  A1 B1 + A1 B2 + A2 B1          (three kind::f16 MMAs into one fp32 TMEM accumulator;
//                                              the dropped A2 B2 term is 2^-22 relative)
// Why fp16 pairs and not bf16 triples: 3 x bf16 needs six products for the same accuracy and three operand
// images; measured in numpy on a 512 x 512 layer (fp64 reference, norm-wise): one bf16 product 2.3e-3, bf16x3 with
// 3 / 6 products 4.4e-6 / 6e-9, plain fp32 2.9e-7 -- the 1e-5 bar of north_star needs the 6-product form or the
// fp16 pair.  fp16's narrow exponent is handled with exact power-of-two scales (operands are multiplied before the
// split, the accumulator divided after; conversions saturate).
//
// One CTA computes a 128 x NT tile (NT <= 256).  Roles: warp 0 streams the pre-split, pre-swizzled weight tiles
// with cp.async.bulk; warp 1 issues the MMAs; warp 2 owns the TMEM allocation; warps 4-11 first LOAD the fp32 A
// tile, split it and store both pieces into the 128B-swizzled operand stage (generic-proxy stores + proxy fence),
// then run the epilogue (bias + exact activation + act', or (.) act', or plain) from TMEM to fp32 global memory.
#include <cuda_fp16.h>

#include <cmath>
#include <cstring>

#include "best_internal.h"
#include "tc_ptx.cuh"

namespace best {
namespace tc32 {

constexpr int BM = 128, BK = 64;
constexpr int kStages = 3;
constexpr int kNT = 128;                        // widest tile: four 128-column accumulators fill the 512 TMEM columns
constexpr int kAStage = 2 * BM * BK * 2;        // two fp16 pieces of 128 x 64: 32 KB
constexpr int kBStage = 2 * kNT * BK * 2;       // two fp16 pieces of <= 128 x 64: 32 KB
constexpr int kThreads = 384;                   // 4 control warps + 8 loader / epilogue warps
constexpr int kWorkers = 256;
enum { EPI_FWD_ACT = 0, EPI_BWD_MUL = 1, EPI_PLAIN = 2 };

struct Smem {
  static constexpr int A = 0;
  static constexpr int B = A + kStages * kAStage;
  static constexpr int BARS = B + kStages * kBStage;   // full_a[3] full_b[3] empty[3] d_full
  static constexpr int TMEMPTR = BARS + 10 * 8;
  static constexpr int TOTAL = TMEMPTR + 16;
};

struct Gemm {
  const float* A; int lda;        // fp32 activations [M][lda]
  const uint8_t* Bpack;           // [n-tile][k-chunk][piece][NT rows][128 B], swizzled, pre-scaled by b_scale
  float* C; int ldc;              // fp32 out [M][ldc]
  int M, N, K, NT;                // NT = tile width (multiple of 16, <= 128)
  const float* bias;              // FWD: [N]
  float* aux; int ldaux;          // FWD: act' out; BWD: act' in
  int act;
  float a_scale, out_scale;       // a is multiplied by a_scale before the split; acc * out_scale = A B
};

__host__ __device__ constexpr uint32_t idesc_f16(int M, int N) {   // kind::f16, A = B = fp16, D = fp32, K-major both
  return (1u << 4) | (0u << 7) | (0u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

__device__ __forceinline__ uint32_t cvt_f16x2_sat(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ void split2(float x0, float x1, uint32_t& h1, uint32_t& h2) {
  h1 = cvt_f16x2_sat(x0, x1);
  const __half2 hh = *reinterpret_cast<const __half2*>(&h1);
  const float2 f = __half22float2(hh);
  h2 = cvt_f16x2_sat(x0 - f.x, x1 - f.y);
}

__device__ __forceinline__ void act_eval(int kind, float a, float& h, float& dh) {
  if (kind == BEST_ACT_TANH) {
    h = tanhf(a);
    dh = 1.0f - h * h;
  } else {  // SiLU, sigma evaluated overflow-safe; ex2-based exp (2 ulp) and a correctly rounded reciprocal: the
            // IEEE divisions of the FFMA path cost 11 k cycles per 64-column sub-tile here
    const float e = __expf(-fabsf(a));
    const float r = __frcp_rn(1.0f + e);
    const float sg = (a >= 0.0f) ? r : e * r;
    h = a * sg;
    dh = sg * (1.0f + a * (1.0f - sg));
  }
}

template <int EPI>
__global__ void __launch_bounds__(kThreads, 1) k_gemm(const Gemm G) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t sbase = ptx::smem_u32(smem);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t bar = sbase + Smem::BARS;
  auto full_a = [&](int s) { return bar + 8u * s; };
  auto full_b = [&](int s) { return bar + 8u * (3 + s); };
  auto empty = [&](int s) { return bar + 8u * (6 + s); };
  const uint32_t d_full = bar + 8u * 9;
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + Smem::TMEMPTR);
  const int m0 = blockIdx.x * BM, nt = blockIdx.y, n0 = nt * G.NT;
  const int kch = (G.K + BK - 1) / BK;
  const uint32_t b_bytes = (uint32_t)G.NT * 256u;   // two pieces of NT rows x 128 B

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) {
      ptx::mbar_init(full_a(s), kWorkers);
      ptx::mbar_init(full_b(s), 1);
      ptx::mbar_init(empty(s), 1);
    }
    ptx::mbar_init(d_full, 1);
    ptx::fence_mbar_init();
  }
  if (warp == 2) ptx::tmem_alloc(sbase + Smem::TMEMPTR, 512);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_ptr;

  if (warp == 0) {
    // ---- weight producer -------------------------------------------------------------------------------
    const uint8_t* src = G.Bpack + (size_t)nt * kch * b_bytes;
    for (int j = 0; j < kch; ++j) {
      const int s = j % kStages, use = j / kStages;
      ptx::mbar_wait(empty(s), (use & 1) ^ 1);
      if (lane == 0) {
        ptx::mbar_arrive_expect_tx(full_b(s), b_bytes);
        ptx::bulk_g2s(sbase + Smem::B + s * kBStage, src + (size_t)j * b_bytes, b_bytes, full_b(s));
      }
      __syncwarp();
    }
  } else if (warp == 1) {
    // ---- MMA issuer: per 64-wide k-chunk 4 K-steps x (A1 B1 + A1 B2 + A2 B1) -----------------------------
    // The tensor core adds into the fp32 accumulator with truncation: the error grows with the NUMBER of
    // accumulations into one accumulator (measured: 96 per accumulator at K = 512 gave 1e-5 relative on the MLP
    // output, the corrections in an accumulator of their own 3e-6).  So the main products of chunk j go to
    // accumulator j mod 3 and the two correction products to a fourth; the epilogue adds the four in fp32.
    const uint32_t idesc = idesc_f16(BM, G.NT);
    const uint32_t b_piece16 = ((uint32_t)G.NT * 128u) >> 4;   // second weight piece, in descriptor units
    for (int j = 0; j < kch; ++j) {
      const int s = j % kStages, use = j / kStages;
      ptx::mbar_wait(full_a(s), use & 1);
      ptx::mbar_wait(full_b(s), use & 1);
      ptx::tc_fence_after();
      if (lane == 0) {
        const uint64_t a1 = ptx::smem_desc_sw128(sbase + Smem::A + s * kAStage);
        const uint64_t a2 = a1 + (uint64_t)((BM * 128) >> 4);
        const uint64_t b1 = ptx::smem_desc_sw128(sbase + Smem::B + s * kBStage);
        const uint64_t b2 = b1 + b_piece16;
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          ptx::mma_bf16_ss(tmem_base + (uint32_t)(j % 3) * kNT, a1 + 2 * kk, b1 + 2 * kk, idesc, (j >= 3 || kk != 0) ? 1u : 0u);
          ptx::mma_bf16_ss(tmem_base + 3u * kNT, a1 + 2 * kk, b2 + 2 * kk, idesc, (j | kk) != 0 ? 1u : 0u);
          ptx::mma_bf16_ss(tmem_base + 3u * kNT, a2 + 2 * kk, b1 + 2 * kk, idesc, 1u);
        }
        ptx::mma_commit(empty(s));
        if (j == kch - 1) ptx::mma_commit(d_full);
      }
      __syncwarp();
    }
  } else if (warp >= 4) {
    // ---- A loader: fp32 rows -> two fp16 pieces in the swizzled stage --------------------------------------
    // 16 lanes read one row's 256-byte chunk (coalesced), a warp two rows per instruction; the loads of the next
    // chunk are issued before waiting for its stage, so the L2 latency hides behind the current chunk's MMAs
    const int wt = tid - 128;              // 0..255
    const int q4 = wt & 15, r0 = wt >> 4;  // 4-column group inside the chunk; first row (rows r0 + 16 i)
    float4 v[2][8];                         // two chunks of loads in flight (L2 latency ~ one chunk's MMA time)
    auto load_chunk = [&](int j, float4 (&dst)[8]) {
      const int k0 = j * BK + q4 * 4;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int r = r0 + 16 * i;
        dst[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (m0 + r < G.M && k0 < G.K) dst[i] = *reinterpret_cast<const float4*>(G.A + (size_t)(m0 + r) * G.lda + k0);
      }
    };
    auto stage_chunk = [&](int s, const float4 (&src)[8]) {
      const uint32_t p1 = sbase + Smem::A + s * kAStage, p2 = p1 + BM * 128;
      const float sc = G.a_scale;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const int r = r0 + 16 * i;
        uint32_t h1[2], h2[2];
        split2(src[i].x * sc, src[i].y * sc, h1[0], h2[0]);
        split2(src[i].z * sc, src[i].w * sc, h1[1], h2[1]);
        const uint32_t off = (uint32_t)r * 128u + (uint32_t)(((q4 >> 1) ^ (r & 7)) << 4) + (uint32_t)(q4 & 1) * 8u;
        ptx::sts_64(p1 + off, ptx::pack2u(h1[0], h1[1]));
        ptx::sts_64(p2 + off, ptx::pack2u(h2[0], h2[1]));
      }
    };
    load_chunk(0, v[0]);
    if (kch > 1) load_chunk(1, v[1]);
    for (int j = 0; j < kch; j += 2) {      // unrolled by two so that the register sets are addressed statically
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int jj = j + u;
        if (jj < kch) {
          const int s = jj % kStages, use = jj / kStages;
          ptx::mbar_wait(empty(s), (use & 1) ^ 1);
          stage_chunk(s, v[u]);
          if (jj + 2 < kch) load_chunk(jj + 2, v[u]);
          ptx::fence_proxy_async();
          ptx::mbar_arrive(full_a(s));
        }
      }
    }
    // ---- epilogue, 64 columns at a time: TMEM (lane = row) -> registers -> math -> shared-memory staging ->
    // global memory by rows.  (Storing straight from the row-per-lane layout writes 16 bytes per 2 KB-strided row
    // and instruction: half-filled sectors, measured 2.5x slower on the whole GEMM.)  The operand stages are free:
    // d_full says every MMA has completed.
    ptx::mbar_wait(d_full, 0);
    ptx::tc_fence_after();
    constexpr int kPitch = 68;                       // floats per staged row: 16-byte stores by rows are conflict-free
    float* stC = reinterpret_cast<float*>(smem + Smem::A);
    float* stD = stC + BM * kPitch;
    const int q = warp & 3, ch = (warp - 4) >> 2;    // TMEM lane quarter; 32-column half of the 64-column sub-tile
    const int row = q * 32 + lane;
    const uint32_t tl = tmem_base + ((uint32_t)(q * 32) << 16);
    const int cw = (warp - 4) * 2 + (lane >> 4), c4 = (lane & 15) * 4;   // row-wise copies: a warp moves 2 rows x 256 B
    const int nsub = (G.NT + 63) >> 6;
    for (int sb = 0; sb < nsub; ++sb) {
      const int nb = n0 + sb * 64;                   // first global column of the sub-tile
      if (EPI == EPI_BWD_MUL) {                      // act' of the sub-tile, by rows
#pragma unroll
        for (int it = 0; it < 8; ++it) {
          const int r = it * 16 + cw;
          float4 d4 = make_float4(0.f, 0.f, 0.f, 0.f);
          if (m0 + r < G.M && nb + c4 < G.N) d4 = *reinterpret_cast<const float4*>(G.aux + (size_t)(m0 + r) * G.ldaux + nb + c4);
          *reinterpret_cast<float4*>(stD + r * kPitch + c4) = d4;
        }
        ptx::named_bar_sync(1, kWorkers);
      }
#pragma unroll
      for (int gg = 0; gg < 2; ++gg) {
        const int cs = ch * 32 + gg * 16;            // column inside the sub-tile
        const int ct = sb * 64 + cs;                 // column inside the tile = TMEM column
        if (ct < G.NT) {
          uint32_t v[16], vc[16], v1[16], v2[16];
          ptx::tmem_ld16(tl + ct, v);
          ptx::tmem_ld16(tl + 3u * kNT + ct, vc);
          if (kch > 1) ptx::tmem_ld16(tl + 1u * kNT + ct, v1);   // (an accumulator no chunk went to holds garbage)
          if (kch > 2) ptx::tmem_ld16(tl + 2u * kNT + ct, v2);
          ptx::tmem_ld_wait();
          float o[16], dv[16];
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            float acc = __uint_as_float(v[i]);
            if (kch > 1) acc += __uint_as_float(v1[i]);
            if (kch > 2) acc += __uint_as_float(v2[i]);
            o[i] = (acc + __uint_as_float(vc[i])) * G.out_scale;
          }
          if (EPI == EPI_FWD_ACT) {
#pragma unroll
            for (int i = 0; i < 16; ++i) {
              const float a = o[i] + ((nb + cs + i < G.N) ? G.bias[nb + cs + i] : 0.0f);
              act_eval(G.act, a, o[i], dv[i]);
            }
          } else if (EPI == EPI_BWD_MUL) {
#pragma unroll
            for (int i4 = 0; i4 < 4; ++i4) {
              const float4 d4 = *reinterpret_cast<const float4*>(stD + row * kPitch + cs + 4 * i4);
              o[4 * i4] *= d4.x; o[4 * i4 + 1] *= d4.y; o[4 * i4 + 2] *= d4.z; o[4 * i4 + 3] *= d4.w;
            }
          }
#pragma unroll
          for (int i4 = 0; i4 < 4; ++i4) {
            *reinterpret_cast<float4*>(stC + row * kPitch + cs + 4 * i4) = make_float4(o[4 * i4], o[4 * i4 + 1], o[4 * i4 + 2], o[4 * i4 + 3]);
            if (EPI == EPI_FWD_ACT)
              *reinterpret_cast<float4*>(stD + row * kPitch + cs + 4 * i4) = make_float4(dv[4 * i4], dv[4 * i4 + 1], dv[4 * i4 + 2], dv[4 * i4 + 3]);
          }
        }
      }
      ptx::named_bar_sync(1, kWorkers);
#pragma unroll
      for (int it = 0; it < 8; ++it) {               // N, ldc, ldaux are multiples of 4 (zero-padded widths)
        const int r = it * 16 + cw;
        if (m0 + r < G.M && nb + c4 < G.N && sb * 64 + c4 < G.NT) {
          *reinterpret_cast<float4*>(G.C + (size_t)(m0 + r) * G.ldc + nb + c4) = *reinterpret_cast<const float4*>(stC + r * kPitch + c4);
          if (EPI == EPI_FWD_ACT)
            *reinterpret_cast<float4*>(G.aux + (size_t)(m0 + r) * G.ldaux + nb + c4) = *reinterpret_cast<const float4*>(stD + r * kPitch + c4);
        }
      }
      ptx::named_bar_sync(1, kWorkers);
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) ptx::tmem_dealloc(tmem_base, 512);
}

}  // namespace tc32
}  // namespace best

// =================================================================================================
// host side: weight packs (split, scaled, swizzled once at best_create) and the per-evaluation launch chain
// =================================================================================================
namespace best {

struct Tc32Op {
  uint8_t* pack = nullptr;   // device
  int N = 0, K = 0, NT = 0;
  float b_scale = 1.0f;
};
struct Tc32Plan {
  std::vector<Tc32Op> fwd;   // fwd[k]: h_k = act(W_k h_{k-1} + b_k), k = 0..nh-1
  std::vector<Tc32Op> bwd;   // bwd[k]: delta_{k-1} = delta_k W_k, k = 1..nh-1;  bwd[0]: grad = delta_0 W_0
};

namespace {

uint16_t f32_to_f16_host(float f) { return __half_as_ushort(__float2half_rn(f)); }
float f16_to_f32_host(uint16_t h) { return __half2float(__ushort_as_half(h)); }

// B[n][k] (logical, n < N, k < K; zero outside) -> [n-tile][k-chunk][piece][NT][128 B] with the 128-byte swizzle
int build_pack(Tc32Op& op, int N, int K, const std::vector<float>& Bm /* [N][K] row-major */) {
  op.N = N; op.K = K;
  op.NT = N >= tc32::kNT ? tc32::kNT : ((N + 15) / 16) * 16;
  float mx = 0.0f;
  for (float v : Bm) mx = std::fmax(mx, std::fabs(v));
  // largest power of two <= 256 that keeps |w| * scale well inside fp16 (65504)
  float sc = 256.0f;
  while (sc > 1.0f / 65536.0f && mx * sc > 16384.0f) sc *= 0.5f;
  op.b_scale = sc;
  const int n_nt = (N + op.NT - 1) / op.NT, kch = (K + tc32::BK - 1) / tc32::BK;
  const size_t tile = (size_t)op.NT * 128;   // bytes of one piece of one (n-tile, k-chunk)
  std::vector<uint16_t> pack((size_t)n_nt * kch * 2 * tile / 2, 0);
  for (int t = 0; t < n_nt; ++t)
    for (int j = 0; j < kch; ++j) {
      uint16_t* base = pack.data() + ((size_t)t * kch + j) * 2 * tile / 2;
      for (int r = 0; r < op.NT; ++r)
        for (int kk = 0; kk < tc32::BK; ++kk) {
          const int n = t * op.NT + r, k = j * tc32::BK + kk;
          const float w = (n < N && k < K) ? Bm[(size_t)n * K + k] * sc : 0.0f;
          const uint16_t h1 = f32_to_f16_host(w);
          const uint16_t h2 = f32_to_f16_host(w - f16_to_f32_host(h1));
          const size_t off = ((size_t)r * 128 + ((((size_t)(kk >> 3)) ^ (size_t)(r & 7)) << 4) + (size_t)(kk & 7) * 2) / 2;
          base[off] = h1;
          base[tile / 2 + off] = h2;
        }
    }
  BEST_TRY(dev_alloc(&op.pack, pack.size() * 2));
  BEST_CUDA(cudaMemcpy(op.pack, pack.data(), pack.size() * 2, cudaMemcpyHostToDevice));
  return BEST_OK;
}

template <int EPI>
int launch(const tc32::Gemm& G, cudaStream_t s) {
  static std::atomic<bool> attr_set{false};
  const int smem_bytes = tc32::Smem::TOTAL + 1024;
  if (!attr_set.load(std::memory_order_acquire)) {
    BEST_CUDA(cudaFuncSetAttribute(tc32::k_gemm<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    attr_set.store(true, std::memory_order_release);
  }
  dim3 grid((G.M + tc32::BM - 1) / tc32::BM, (G.N + G.NT - 1) / G.NT);
  tc32::k_gemm<EPI><<<grid, tc32::kThreads, smem_bytes, s>>>(G);
  count_launch();
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

}  // namespace

// W_flat / b_flat as in best_config.  ctx->W / ctx->b (padded fp32 copies) stay for the biases and the output layer.
int tc32_plan_create(best_ctx* ctx, const best_config* cfg) {
  const int nh = cfg->n_affine - 1;
  if (nh < 1) { set_error("BEST_PREC_FP32_TC needs at least one hidden layer"); return BEST_ERR_UNSUPPORTED; }
  for (int k = 1; k <= nh; ++k)
    if (cfg->widths[k] < 64) { set_error("BEST_PREC_FP32_TC: hidden widths must be >= 64"); return BEST_ERR_UNSUPPORTED; }
  Tc32Plan* pl = new Tc32Plan();
  ctx->tc32 = pl;
  pl->fwd.resize(nh);
  pl->bwd.resize(nh);
  size_t wo = 0;
  for (int k = 0; k < nh; ++k) {
    const int nin = cfg->widths[k], nout = cfg->widths[k + 1];
    const int pin = ctx->wp[k], pout = ctx->wp[k + 1];
    std::vector<float> F((size_t)pout * pin, 0.0f), Bt((size_t)pin * pout, 0.0f);
    for (int r = 0; r < nout; ++r)
      for (int c = 0; c < nin; ++c) {
        const float w = cfg->W_flat[wo + (size_t)r * nin + c];
        F[(size_t)r * pin + c] = w;      // forward: B[n = out][k = in]
        Bt[(size_t)c * pout + r] = w;    // backward: B[n = in][k = out]
      }
    BEST_TRY(build_pack(pl->fwd[k], pout, pin, F));
    BEST_TRY(build_pack(pl->bwd[k], pin, pout, Bt));
    wo += (size_t)nin * nout;
  }
  return BEST_OK;
}

void tc32_plan_destroy(best_ctx* ctx) {
  Tc32Plan* pl = ctx->tc32;
  if (!pl) return;
  for (auto& o : pl->fwd) cudaFree(o.pack);
  for (auto& o : pl->bwd) cudaFree(o.pack);
  delete pl;
  ctx->tc32 = nullptr;
}

// C = epi(A B) for one layer; shapes as in emulator_fp32.cu's launch_gemm
int tc32_gemm(best_ctx* ctx, bool forward, int layer, const float* A, int lda, float* C, int ldc, int M,
              const float* bias, float* aux, int ldaux, int epi, cudaStream_t s) {
  const Tc32Op& op = forward ? ctx->tc32->fwd[layer] : ctx->tc32->bwd[layer];
  tc32::Gemm G{};
  G.A = A; G.lda = lda; G.Bpack = op.pack; G.C = C; G.ldc = ldc;
  G.M = M; G.N = op.N; G.K = op.K; G.NT = op.NT;
  G.bias = bias; G.aux = aux; G.ldaux = ldaux; G.act = ctx->activation;
  // activations: x16 (|h| up to 4e3 before the conversion saturates); deltas are small: x4096
  G.a_scale = forward ? 16.0f : 4096.0f;
  G.out_scale = 1.0f / (G.a_scale * op.b_scale);
  switch (epi) {
    case tc32::EPI_FWD_ACT: return launch<tc32::EPI_FWD_ACT>(G, s);
    case tc32::EPI_BWD_MUL: return launch<tc32::EPI_BWD_MUL>(G, s);
    default: return launch<tc32::EPI_PLAIN>(G, s);
  }
}

}  // namespace best
