// bf16 tensor-core path (BEST_PREC_BF16): ONE persistent kernel per best_step_* call.
//
// A CTA owns a tile of 128 chains for all n_steps.  TMEM lane r == chain r:
//   warp 0 (1 lane)  weight producer: streams pre-swizzled bf16 weight tiles L2 -> SMEM ring with
//                    cp.async.bulk + mbarrier complete_tx (weights are packed once at best_create)
//   warp 1 (1 lane)  MMA issuer: tcgen05.mma.cta_group::1.kind::f16, M=128, N<=256, K=16;
//                    A = activations resident in SMEM (128B swizzle, written in place by the
//                    epilogue), B = weight stage (64B swizzle), D = fp32 in TMEM (2 x 256 columns)
//   warp 2           TMEM allocation
//   warps 4-19       four threads per chain (one per warp of the chain's TMEM lane quarter):
//                    tcgen05.ld epilogues (bias + activation + act' / delta) on 16 of every 64
//                    columns each, and cooperatively Philox, whitened proposal, Gaussian / banana /
//                    box terms and the accept decision on 8 parameter dimensions each.
// ROWS = 256 (the default for 512-wide layers at >= 9.5 k chains) runs the same tile on a CTA PAIR: cta_group::2
// MMAs with M = 256, each CTA staging half of every weight tile (Geo<256>).
// The MLP forward and its input-gradient backprop (A1b, A1c) are a chain of GEMMs whose
// activations never leave the SM; only act' (bf16) is parked in an L2-resident scratch between
// the forward and backward sweeps.  See DESIGN.md §"tensor-core kernel".
#include <cuda.h>

#include <algorithm>
#include <cstdlib>
#include <cstring>

#include "device_math.cuh"
#include "tc_fused.h"
#include "tc_ptx.cuh"

namespace best {

namespace tc {

constexpr int kRows = 128;           // TMEM lanes == MMA M
// Tile geometries (template parameter ROWS of the kernel = chains per CTA):
//   ROWS = 128 : 128 chains per CTA, hidden width <= 512.  A k-chunk = 128 rows x 64 bf16 = 16 KB;
//                the epilogue rewrites the activation operand IN PLACE (a full layer of fp32
//                accumulators, 128 x 512, is exactly the 512 TMEM columns).
//   ROWS = 64 / 32: fewer chains per CTA (1024-wide layers, or batches too small to fill 148 SMs
//                with 128-chain tiles).  A k-chunk = ROWS x 64 bf16 at a ROWS x 128 B pitch, so
//                that the MMA (still M = 128) reads the FOLLOWING chunks as rows ROWS..127:
//                phantom rows whose accumulator lanes nobody reads.  A layer of
//                accumulators (1024 columns) no longer fits TMEM, so the epilogue writes the
//                next operand to an L2-resident image and warp 3 copies it back chunk by chunk
//                (cp.async.bulk) as soon as the last N-chunk's MMAs have released the chunk.
//   ROWS = 264 : CTA PAIR for 1024-wide layers (cluster of 2, tcgen05 cta_group::2): 64 chains per CTA,
//                the leader CTA issues M = 128 MMAs over both CTAs' rows, each CTA streams HALF of
//                every weight tile, and an N = 256 accumulator chunk takes only 128 TMEM columns per
//                CTA (lanes 64..127 hold the upper half of N for the same 64 rows), so a whole
//                1024-wide layer of accumulators fits TMEM and the operand is rewritten in place.
template <int ROWS> struct Geo {
  static_assert(ROWS == 128 || ROWS == 64 || ROWS == 32 || ROWS == 264 || ROWS == 265 || ROWS == 233 || ROWS == 232 || ROWS == 256, "tile geometry");
  static constexpr bool kPair = (ROWS == 264 || ROWS == 265 || ROWS == 233 || ROWS == 232);
  // ROWS = 256: geometry 128 on a CTA PAIR (cluster of 2, tcgen05 cta_group::2 with M = 256): 128 chains per CTA,
  // lane = chain and all N columns in the CTA's own TMEM exactly as in geometry 128, but the leader issues ONE MMA
  // for both CTAs' rows and each CTA stages only HALF of every weight tile.  A 128 x 256 x 16 bf16 MMA from shared
  // memory reads 4 KB of A and 8 KB of B per 128 cycles = 96 B/cycle of the SM's 128 B/cycle shared-memory port;
  // with B split over the pair it is 64 B/cycle, which leaves the epilogue's loads and stores room
  // (profiles/r2b), and the L2 -> SM weight stream halves.
  static constexpr bool kWide = (ROWS == 256);
  static constexpr bool kCluster = kPair || kWide;   // cluster of two CTAs, leader issues, peer arrives remotely
  // ROWS = 232: geometry 264 (1024-wide, in place) with 32 chains per CTA, the compact operand (16 chunks at a
  // 4 KB pitch = 64 KB) and the 8-stage weight ring of geometry 233 -- for batches that leave SMs idle with
  // 64-chain CTAs (the small points of the configs[4] sweep).
  static constexpr bool kHalf = (ROWS == 233 || ROWS == 232);   // 32 chains in the CTA's 64 MMA rows
  // ROWS = 265: CTA pair for 512-wide layers.  64 chains per CTA need only 64 KB of operand and 256
  // TMEM columns per layer, so BOTH are double-buffered: an op reads operand buffer (op & 1) and its
  // epilogue writes the other one, accumulators alternate between two sets of TMEM columns.  No
  // in-place hazard is left: the next op's MMAs start on the first finished k-chunk while this op's
  // epilogue is still running.
  // ROWS = 233: geometry 265 with only 32 CHAINS per CTA (rows 32..63 of the CTA's 64 MMA rows are phantom:
  // never written, their accumulator lanes never read).  The epilogue warps of the phantom row quarter do
  // nothing at all, so the 8 working warps have two issue slots per scheduler cycle pair to themselves and a
  // batch too small to fill the chip with 64-chain CTAs (4096 chains = 64 CTAs) spreads over twice the SMs.
  static constexpr bool kPingPong = (ROWS == 265 || ROWS == 233);
  static constexpr bool kInPlace = (ROWS == 128 || kPair || kWide);   // operand stays in SMEM
  // ROWS = 128 / 256, every N-chunk but the last of an op: each 64-column k-chunk of the next operand is produced by ONE
  // of a row's four epilogue threads (warp k owns the groups grp = k mod 4 and walks them in four 16-column
  // pieces), so the store -> proxy fence -> arrive sequence is paid once per 64 columns of a thread instead of
  // once per 16; the owner arrives on a_ready for all four.  The LAST N-chunk keeps the interleaved order (all
  // four threads on the same group): the next op's MMAs wait for exactly these k-chunks, one after the other.
  static constexpr bool kOwn = (ROWS == 128 || ROWS == 256);
  static constexpr bool kOwnLastInterleaved = true;
  static constexpr int kTileRows = kPair ? 64 : (kWide ? 128 : ROWS);   // rows of the CTA's operand / act' blocks
  static constexpr int kChains = kHalf ? 32 : kTileRows;   // chains the CTA advances
  static constexpr int kEpiArrive = kHalf ? 256 : 512;      // epilogue threads that run (per CTA)
  // bytes between consecutive 64-column k-chunks of the operand.  Geometry 233 keeps only its 32 real rows:
  // the MMA reads the following chunk's rows as its phantom rows 32..63 (finite bf16 of the same chain tile or
  // weight-ring bytes; their accumulator lanes are never read), which halves the operand buffers (2 x 32 KB)
  // and leaves room for an 8-stage weight ring: four stages in flight cover only ~450 cycles per stage of
  // the L2 latency, measured as the issue rate of the N-chunk-outer order.
  static constexpr int kAChunk = kHalf ? 4096 : kTileRows * 128;
  static constexpr int kPPStride = (ROWS == 233) ? 32768 : 65536;   // ping-pong: bytes between the two operand buffers
  static constexpr int kStagesOff = kHalf ? 65536 : 131072; // weight ring: offset in the carve-up (SmemLayout::STAGES)
  static constexpr int kEpiActive = kPair ? 512 : kTileRows * 4;   // epilogue threads with MLP epilogue work
  static constexpr int kNBuf = kPair ? 4 : 2;          // accumulator buffers
  static constexpr int kBufCols = kPair ? 128 : 256;   // TMEM columns per buffer
  static constexpr int kStagesG = kHalf ? 8 : 4;   // weight ring: stages
  static constexpr int kStageBytesG = 16384;           // ... of this many bytes per CTA (pair: one K = 64 slice)
};
constexpr int kAChunkBytes = 16384;  // R64 = false chunk pitch (also the exchange-slot size)
constexpr int kMaxKch = 16;          // hidden width <= 1024
constexpr int kStageBytes = 16384;   // weight stage: <=256 rows x 32 bf16 (64 B rows, SW64)
constexpr int kStages = 4;
constexpr int kMaxOps = 12;
constexpr int kCtrlWarps = 4;          // producer, MMA issuer, TMEM allocator, spare
constexpr int kEpiWarps = 16;          // 4 per TMEM lane quarter
constexpr int kThreads = (kCtrlWarps + kEpiWarps) * 32;
constexpr int kDP = 32;              // parameter vectors are padded to 32 inside the kernel

enum { EPI_FWD_HID = 0, EPI_FWD_LAST = 1, EPI_BWD_HID = 2, EPI_BWD_FINAL = 3 };
enum { M_MH = 0, M_MALA = 1, M_HMC = 2, M_AIES = 3, M_EVAL = 4 };
enum { IO_ROWS_F32 = 0, IO_SOA_F64 = 1 };

struct OpDesc {
  int kch;    // 64-wide k-chunks of the A operand
  int nch;    // n-chunks (each one TMEM buffer)
  int ncols;  // columns per n-chunk (MMA N)
  int epi;
  int layer;  // FWD: hidden layer index (0-based) whose bias/act is applied; BWD_HID: layer whose act' multiplies
  int paired; // CTA-pair kernel, 1024-wide: N-chunks are issued two at a time, k-chunk outer (see mma_loop_pair)
  int perm;   // CTA-pair kernels: the four 64-row blocks of a B chunk are packed 0,2,1,3 (see pair_jn)
};

struct Params {
  // CTA-pair kernel: the weight pack as a 2-D byte tensor [rows][256 B], boxes of 32 rows (8 KB) / 4 rows (1 KB)
  CUtensorMap wmap8, wmap1;
  int d, H, n_hidden, act;
  float mlp_scale, b_out;
  int n_ops_fwd, n_ops_all;
  OpDesc ops[kMaxOps];
  const uint8_t* wpack;   // packed tiles: forward ops then backward ops, consumption order
  const float* bias;      // [n_hidden][H] fp32 (bias16: staged in SMEM as bf16, 2 per word)
  const float* w_out;     // [H]
  uint16_t* dact;         // scratch: per tile [n_hidden-1][H/64][8 pieces][tile rows][8] bf16
  size_t dact_tile_elems;
  uint8_t* aimg;          // ROWS < 128: per tile, SMEM image of the next A operand [16 chunks][ROWS][128 B]
  int kch_max;            // k-chunks of the widest operand (= H / 64): barriers 0..kch_max-1 are in use
  int bias16;             // bias table kept as bf16 in SMEM (1024-wide layers)
  // target terms (fp64 masters on device, converted to fp32 in SMEM at kernel start)
  int has_gauss, has_box, banana_i, banana_j;
  int hard_box;   // set per launch from the context (8(f)#1)
  float banana_sigma, pen_kappa, pen_gamma;
  const double *mu, *R, *lo, *hi, *L;
};

struct Run {
  int method, want_grad, io_mode;
  int64_t B;            // chains (or points) covered by this launch
  int64_t ld;           // leading dimension of the SoA state arrays
  int64_t n_steps;
  uint64_t step0, seed;
  float eps;            // MH/MALA/HMC step size; AIES: a
  int n_leapfrog;
  // state (fp64 SoA [d][ld])
  double *theta, *grad, *logp, *last_la;
  unsigned long long* n_accept;
  // EVAL i/o
  const float* in_rows; float* out_logp; float* out_grad;
  // AIES
  int64_t own0, oth0;
  int64_t n_oth;        // walkers of the other half (partner range); = B unless the ensemble is sharded over ranks
  int de;               // differential-evolution move (eq 2.16) instead of the stretch move; eps = sigma_gamma
  // Philox chain id = chain0 + chain index (multi-GPU shards draw disjoint streams)
  uint32_t chain0;
  // A8: post-accept theta written by the kernel itself, fp32 rows [slot][B_rows][d]:
  //   trace: slot (t_call0 + t + 1) / thin - 1 whenever thin divides t_call0 + t + 1 (t = step inside this launch);
  //   win:   slot t, every step (the covariance window buffer of A9)
  float* trace; int thin; int64_t t_call0;
  float* win;
  int64_t B_rows;       // chains per trace / window slot (= the state's chain count)
  // EVAL only: tiles of the whole call.  The grid holds at most one wave of CTAs (pairs); CTA b evaluates tiles
  // b, b + gridDim.x, ... in one launch, so prologue, TMEM allocation and launch are paid once per CTA, not per tile
  int64_t n_tiles;
};

// shared-memory carve-up (dynamic, 1024-byte aligned base)
struct SmemLayout {
  static constexpr int A = 0;
  static constexpr int STAGES = A + 131072;                          // 8 x 16 KB or 16 x 8 KB chunks
  static constexpr int BIAS = STAGES + kStages * kStageBytes;        // 196608: 2048 floats / 4096 bf16
  static constexpr int WOUTS = BIAS + 2048 * 4;                      // 1024 floats (s * w_out)
  static constexpr int LMAT = WOUTS + 1024 * 4;                      // 32x32 floats
  static constexpr int LTMAT = LMAT + 1024 * 4;                      // L transposed
  static constexpr int RMAT = LTMAT + 1024 * 4;
  static constexpr int RTMAT = RMAT + 1024 * 4;
  static constexpr int VECS = RTMAT + 1024 * 4;                      // mu, lo, hi, 1/width: 4x32 floats
  static constexpr int PART = VECS + 4 * 32 * 4;                     // partial sums [2][4][128] floats
  static constexpr int BARS = PART + 2 * 4 * 128 * 4;
  // barriers: full[8] empty[8] a_ready[16] a_free[16] d_full[4] d_free[4] epi_done[4] xin_done
  static constexpr int NBARS = 61;
  static constexpr int TMEMPTR = BARS + NBARS * 8;
  static constexpr int TOTAL = TMEMPTR + 16;
};
static_assert(SmemLayout::TOTAL + 1024 <= 232448, "shared memory budget");
static_assert(Geo<265>::kStagesOff == SmemLayout::STAGES && Geo<128>::kStagesOff == SmemLayout::STAGES &&
              Geo<256>::kStagesOff == SmemLayout::STAGES, "weight ring offset");
static_assert(Geo<233>::kStagesOff + Geo<233>::kStagesG * Geo<233>::kStageBytesG <= SmemLayout::BIAS &&
              Geo<233>::kPPStride + 8 * Geo<233>::kAChunk <= Geo<233>::kStagesOff, "geometry 233 carve-up");
static_assert(16 * Geo<232>::kAChunk <= Geo<232>::kStagesOff, "geometry 232 carve-up");

struct Bars {  // mbarrier addresses are computed, never looked up (keeps them out of local memory)
  uint32_t base;
  __device__ __forceinline__ uint32_t full(int i) const { return base + 8u * i; }
  __device__ __forceinline__ uint32_t empty(int i) const { return base + 8u * (8 + i); }
  __device__ __forceinline__ uint32_t a_ready(int j) const { return base + 8u * (16 + j); }
  __device__ __forceinline__ uint32_t a_free(int j) const { return base + 8u * (32 + j); }
  __device__ __forceinline__ uint32_t d_full(int b) const { return base + 8u * (48 + b); }
  __device__ __forceinline__ uint32_t d_free(int b) const { return base + 8u * (52 + b); }
  __device__ __forceinline__ uint32_t epi_done(int c) const { return base + 8u * (56 + c); }
  __device__ __forceinline__ uint32_t xin_done() const { return base + 8u * 60; }
};
__device__ __forceinline__ Bars make_bars(uint32_t base) { Bars b; b.base = base; return b; }

// ------------------------------------------------------------------------------------------------
// weight producer (warp 0, warp-converged; one elected lane issues the copies)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "elect.sync _|p, 0xffffffff;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(pred));
  return pred != 0;
}

__device__ void producer_loop(const Params& P, const Bars& bars, uint32_t stage_base, int64_t n_evals,
                              int n_ops) {
  uint32_t t = 0;  // running tile counter: stage = t % kStages, use = t / kStages
  for (int64_t e = 0; e < n_evals; ++e) {
    const uint8_t* src = P.wpack;
    for (int oi = 0; oi < n_ops; ++oi) {
      const OpDesc op = P.ops[oi];
      const uint32_t bytes = (uint32_t)op.ncols * 64u;
      const int ntiles = op.nch * op.kch * 2;
      for (int i = 0; i < ntiles; ++i, ++t) {
        const uint32_t s = t % kStages, use = t / kStages;
        ptx::mbar_wait(bars.empty(s), (use & 1u) ^ 1u);
        if (elect_one()) {
          ptx::mbar_arrive_expect_tx(bars.full(s), bytes);
          ptx::bulk_g2s(stage_base + s * kStageBytes, src, bytes, bars.full(s));
        }
        __syncwarp();
        src += bytes;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// MMA issuer (warp 1, warp-converged so that descriptors live in uniform registers; one elected
// lane issues tcgen05.mma / tcgen05.commit)
// ------------------------------------------------------------------------------------------------
template <int ROWS>
__device__ void mma_loop(const Params& P, const Bars& bars, uint32_t a_base, uint32_t stage_base,
                         uint32_t tmem_base, int64_t n_evals, int n_ops) {
  uint32_t t = 0;  // tile counter (mirrors the producer)
  uint32_t g = 0;  // n-chunk counter: TMEM buffer = g & 1
  uint32_t o = 0;  // op counter: phase of a_ready / a_free
  const uint64_t adesc0 = ptx::smem_desc_sw128(a_base);
  const uint64_t bdesc0 = ptx::smem_desc_sw64(stage_base);
  for (int64_t e = 0; e < n_evals; ++e) {
    for (int oi = 0; oi < n_ops; ++oi, ++o) {
      const OpDesc op = P.ops[oi];
      const uint32_t idesc = ptx::idesc_bf16(kRows, op.ncols);
      // chunks this op does not read are free as soon as everything issued so far has completed
      if (elect_one())
        for (int j = op.kch; j < P.kch_max; ++j) ptx::mma_commit(bars.a_free(j));
      __syncwarp();
      for (int c = 0; c < op.nch; ++c, ++g) {
        const uint32_t buf = g & 1u, use = g >> 1;
        ptx::mbar_wait(bars.d_free(buf), (use & 1u) ^ 1u);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + buf * 256u;
        const bool last_c = (c == op.nch - 1);
        for (int j = 0; j < op.kch; ++j) {
          if (c == 0) {
            ptx::mbar_wait(bars.a_ready(j), o & 1u);
            ptx::tc_fence_after();
          }
#pragma unroll
          for (int h = 0; h < 2; ++h, ++t) {
            const uint32_t s = t % kStages, use_s = t / kStages;
            ptx::mbar_wait(bars.full(s), use_s & 1u);
            ptx::tc_fence_after();
            // descriptor start-address fields are in 16-byte units
            const uint64_t ad = adesc0 + (uint64_t)((j * Geo<ROWS>::kAChunk + h * 64) >> 4);
            const uint64_t bd = bdesc0 + (uint64_t)((s * kStageBytes) >> 4);
            if (elect_one()) {
              ptx::mma_bf16_ss(d_tmem, ad, bd, idesc, (j | h) != 0 ? 1u : 0u);
              ptx::mma_bf16_ss(d_tmem, ad + 2, bd + 2, idesc, 1u);
              ptx::mma_commit(bars.empty(s));
              if (last_c && h == 1) ptx::mma_commit(bars.a_free(j));
            }
            __syncwarp();
          }
        }
        if (elect_one()) ptx::mma_commit(bars.d_full(buf));
        __syncwarp();
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// A-operand loader (warp 3, ROWS < 128 only): the only thread that arrives on a_ready.  Per evaluation:
// the input chunk written by the sampler threads (xin_done), then after every op but the last the
// 16 chunks of the next operand, copied L2 image -> SMEM as soon as (a) the epilogue has written
// the N-chunk they come from (epi_done) and (b) the current op's MMAs have released them (a_free).
// ------------------------------------------------------------------------------------------------
__device__ void loader_loop(const Params& P, const Bars& bars, uint32_t a_base, const uint8_t* aimg_tile,
                            uint32_t chunk_bytes, int64_t n_evals, int n_ops) {
  uint32_t o = 0;   // op counter (phase of a_ready / a_free / epi_done)
  for (int64_t e = 0; e < n_evals; ++e) {
    ptx::mbar_wait(bars.xin_done(), (uint32_t)(e & 1));
    if (elect_one())
      for (int j = 0; j < P.kch_max; ++j) ptx::mbar_arrive(bars.a_ready(j));
    __syncwarp();
    for (int oi = 0; oi + 1 < n_ops; ++oi, ++o) {
      const OpDesc op = P.ops[oi];
      const int out_kch = (op.nch * op.ncols) >> 6;   // k-chunks of the operand this op produces
      for (int j = 0; j < P.kch_max; ++j) {
        if (j < out_kch) {
          ptx::mbar_wait(bars.epi_done((j * 64) / op.ncols), o & 1u);
          ptx::mbar_wait(bars.a_free(j), o & 1u);
          if (elect_one()) {
            ptx::mbar_arrive_expect_tx(bars.a_ready(j), chunk_bytes);
            ptx::bulk_g2s(a_base + j * chunk_bytes, aimg_tile + (size_t)j * chunk_bytes, chunk_bytes, bars.a_ready(j));
          }
        } else if (elect_one()) {
          ptx::mbar_arrive(bars.a_ready(j));
        }
        __syncwarp();
      }
    }
    ++o;   // the last op of the evaluation produces no operand
  }
}

// ------------------------------------------------------------------------------------------------
// CTA-pair roles (Geo<264>, Geo<265>).  Both CTAs run the producer and the epilogue; the leader (cluster
// rank 0) issues the MMAs.  Every barrier the issuer waits on lives in the LEADER's shared memory: each
// CTA's producer loads its own half of a weight stage with 2-SM tensor copies that credit the leader's
// full barrier, and the peer's epilogue threads arrive on the leader's a_ready / d_free directly
// (shared::cluster address with the rank bit cleared).
// ------------------------------------------------------------------------------------------------
template <int ROWS>
__device__ void producer_loop_pair(const Params& P, const Bars& bars, uint32_t stage_base, uint32_t rank,
                                   int64_t n_evals, int n_ops) {
  constexpr uint32_t NS = Geo<ROWS>::kStagesG, SB = Geo<ROWS>::kStageBytesG;
  uint32_t t = 0;   // stage counter: one stage = one 64-wide k-chunk = two K32 tiles (this CTA's halves)
  for (int64_t e = 0; e < n_evals; ++e) {
    uint32_t src = 0;   // byte offset inside the pack
    for (int oi = 0; oi < n_ops; ++oi) {
      const OpDesc op = P.ops[oi];
      const uint32_t bytes = (uint32_t)op.ncols * 64u, half = bytes >> 1;   // rows [rank N/2, +N/2) of a tile
      const void* tmap = (half == 8192u) ? (const void*)&P.wmap8 : (const void*)&P.wmap1;
      const int nst = op.nch * op.kch;
      for (int i = 0; i < nst; ++i, ++t) {
        const uint32_t s = t % NS, use = t / NS;
        ptx::mbar_wait(bars.empty(s), (use & 1u) ^ 1u);
        if (elect_one()) {
          // all four halves' bytes land on the LEADER's full barrier; only the leader arrives on it
          if (rank == 0) ptx::mbar_arrive_expect_tx(bars.full(s), 2u * bytes);
          ptx::tma_2sm_load_2d(stage_base + s * SB, tmap, bars.full(s), 0, (int)((src + rank * half) >> 8));
          ptx::tma_2sm_load_2d(stage_base + s * SB + half, tmap, bars.full(s), 0, (int)((src + bytes + rank * half) >> 8));
        }
        __syncwarp();
        src += 2u * bytes;
      }
    }
  }
}

// Two warps of the leader CTA issue (wq = 0: warp 1, wq = 1: warp 3).  A pair MMA is only 64 cycles of
// tensor work but costs ~50 cycles to issue (+ the stage wait / commit), so ONE issuer was measured at
// ~450 cycles per 16 KB stage against the 256 the tensor pipe needs; in the paired order the two
// N-chunks of a pass have their own accumulators and their own (alternating) stages, so each warp
// takes one of them.  Ops that are not paired are issued by warp 1 alone.  a_free counts 2 arrivals.
template <bool LEADER, int ROWS>
__device__ void mma_loop_pair(const Params& P, const Bars& bars, uint32_t a_base, uint32_t stage_base,
                              uint32_t tmem_base, int64_t n_evals, int n_ops, int wq) {
  constexpr uint32_t NS = Geo<ROWS>::kStagesG, SB = Geo<ROWS>::kStageBytesG, NB = Geo<ROWS>::kNBuf;
  uint32_t t = 0, g = 0, o = 0;
  const uint64_t adesc0 = ptx::smem_desc_sw128(a_base);
  const uint64_t bdesc0 = ptx::smem_desc_sw64(stage_base);
  for (int64_t e = 0; e < n_evals; ++e) {
    for (int oi = 0; oi < n_ops; ++oi, ++o) {
      const OpDesc op = P.ops[oi];
      const uint32_t idesc = ptx::idesc_bf16(Geo<ROWS>::kWide ? 256 : kRows, op.ncols);
      const uint32_t half16 = ((uint32_t)op.ncols * 32u) >> 4;   // one K32 tile half, in descriptor units
      if (LEADER && wq == 0 && !Geo<ROWS>::kPingPong) {   // (ping-pong: nothing is overwritten in place, a_free unused)
        if (elect_one())
          for (int j = op.kch; j < P.kch_max; ++j) { ptx::mma_commit_2cta(bars.a_free(j)); ptx::mma_commit_2cta(bars.a_free(j)); }
        __syncwarp();
      }
      if (op.paired) {
        // Two N-chunks at a time, k-chunk outer: a_free(j) of the LAST pass then fires while that pass is
        // still running (k-chunk by k-chunk) and the first pass's epilogue overlaps it, instead of every
        // epilogue store waiting for the last N-chunk's sweep over K.
        for (int c = 0; c < op.nch; c += 2, g += 2) {
          const uint32_t b0 = g % NB, b1 = (g + 1) % NB, u0 = g / NB, u1 = (g + 1) / NB;
          const bool last_p = (c + 2 >= op.nch);
          if (LEADER) {
            const uint32_t bq = wq ? b1 : b0, uq = wq ? u1 : u0;
            ptx::mbar_wait(bars.d_free(bq), (uq & 1u) ^ 1u);
            ptx::tc_fence_after();
            const uint32_t d_tmem = tmem_base + bq * Geo<ROWS>::kBufCols;
            for (int j = 0; j < op.kch; ++j) {
              if (c == 0) ptx::mbar_wait(bars.a_ready(j), o & 1u);
              const uint64_t ad = adesc0 + (uint64_t)((j * Geo<ROWS>::kAChunk + (Geo<ROWS>::kPingPong ? (oi & 1) * Geo<ROWS>::kPPStride : 0)) >> 4);
              const uint32_t tt = t + 2u * (uint32_t)j + (uint32_t)wq, s = tt % NS, use_s = tt / NS;
              ptx::mbar_wait(bars.full(s), use_s & 1u);
              ptx::tc_fence_after();
              const uint64_t bd = bdesc0 + (uint64_t)((s * SB) >> 4);
              if (elect_one()) {
                ptx::mma_bf16_ss_2cta(d_tmem, ad, bd, idesc, j != 0 ? 1u : 0u);
                ptx::mma_bf16_ss_2cta(d_tmem, ad + 2, bd + 2, idesc, 1u);
                ptx::mma_bf16_ss_2cta(d_tmem, ad + 4, bd + half16, idesc, 1u);
                ptx::mma_bf16_ss_2cta(d_tmem, ad + 6, bd + half16 + 2, idesc, 1u);
                ptx::mma_commit_2cta(bars.empty(s));
                if (last_p && !Geo<ROWS>::kPingPong) ptx::mma_commit_2cta(bars.a_free(j));   // one arrival per issuing warp
              }
              __syncwarp();
            }
            if (elect_one()) ptx::mma_commit_2cta(bars.d_full(bq));
            __syncwarp();
          }
          t += 2u * (uint32_t)op.kch;
        }
        continue;
      }
      if (wq != 0) {   // not this warp's op: only keep in step with the operand barrier's phases
        if (LEADER) ptx::mbar_wait(bars.a_ready(0), o & 1u);
        t += (uint32_t)(op.nch * op.kch); g += (uint32_t)op.nch;
        continue;
      }
      for (int c = 0; c < op.nch; ++c, ++g) {
        const uint32_t buf = g % NB, use = g / NB;
        if (LEADER) {
          ptx::mbar_wait(bars.d_free(buf), (use & 1u) ^ 1u);   // both CTAs' epilogue threads arrive here
          ptx::tc_fence_after();
        }
        const uint32_t d_tmem = tmem_base + buf * Geo<ROWS>::kBufCols;
        const bool last_c = (c == op.nch - 1);
        for (int j = 0; j < op.kch; ++j, ++t) {
          if (LEADER) {
            if (c == 0) ptx::mbar_wait(bars.a_ready(j), o & 1u);   // both CTAs' k-chunk j
            const uint32_t s = t % NS, use_s = t / NS;
            ptx::mbar_wait(bars.full(s), use_s & 1u);   // both CTAs' halves of both K32 tiles
            ptx::tc_fence_after();
            const uint64_t ad = adesc0 + (uint64_t)((j * Geo<ROWS>::kAChunk + (Geo<ROWS>::kPingPong ? (oi & 1) * Geo<ROWS>::kPPStride : 0)) >> 4);
            const uint64_t bd = bdesc0 + (uint64_t)((s * SB) >> 4);
            if (elect_one()) {
              ptx::mma_bf16_ss_2cta(d_tmem, ad, bd, idesc, j != 0 ? 1u : 0u);
              ptx::mma_bf16_ss_2cta(d_tmem, ad + 2, bd + 2, idesc, 1u);
              ptx::mma_bf16_ss_2cta(d_tmem, ad + 4, bd + half16, idesc, 1u);
              ptx::mma_bf16_ss_2cta(d_tmem, ad + 6, bd + half16 + 2, idesc, 1u);
              ptx::mma_commit_2cta(bars.empty(s));
              if (last_c && !Geo<ROWS>::kPingPong) { ptx::mma_commit_2cta(bars.a_free(j)); ptx::mma_commit_2cta(bars.a_free(j)); }
            }
            __syncwarp();
          }
        }
        if (LEADER) {
          if (elect_one()) ptx::mma_commit_2cta(bars.d_full(buf));
          __syncwarp();
        }
      }
    }
  }
}

}  // namespace tc
}  // namespace best

#include "tc_epilogue.cuh"
#include "tc_host.cuh"
