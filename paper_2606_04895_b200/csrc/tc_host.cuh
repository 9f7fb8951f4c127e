// Kernel body (role dispatch + sampler drivers) and host side (weight packing, launches) of the
// tensor-core path.  Included by tc_fused.cu only.
#pragma once

namespace best {
namespace tc {

// Sampler driver: executed by all 512 epilogue threads; thread (row, k) owns dims [8k, 8k+8) of
// chain `row`.  Scalars (log pi, log alpha, accept) are computed redundantly and identically by the
// four threads of a chain, so they take the same accept branch.
// A8: the post-accept theta of the CTA's chains into row-major fp32 rows [slot][B_rows][d] -- the trace slot of
// this step (every `thin` steps) and / or the covariance window slot (every step).  The rows of a tile are
// contiguous in both, so the sampler threads stage them in shared memory (operand bytes 48-64 KB, dead between
// two evaluations) and ONE thread sends the block with a bulk async copy: direct stores (8 x 4 B per thread at a
// 4d-byte stride across lanes, 32 sectors per instruction) cost ~3.5 k cycles of LSU time per step and SM, measured
// as 2-5 % of a step.  Called by every sampler thread of the CTA (a CTA-wide named barrier inside); `valid` masks
// the ragged tail, `first` is the global index of the tile's first chain inside a slot.  Unaligned blocks (a
// chain count that is not a multiple of 4, an unaligned trace pointer) fall back to direct stores.
template <int ROWS>
__device__ __forceinline__ void emit_tile(EpiCtx& C, const Run& R, int64_t t, int64_t first, int d,
                                          const float (&cur)[8], bool valid) {
  const bool tr_now = R.trace != nullptr && (R.t_call0 + t + 1) % R.thin == 0;
  if (!tr_now && R.win == nullptr) return;   // (uniform over the CTA)
  const int64_t in_launch = (int64_t)blockIdx.x * Geo<ROWS>::kChains;
  int nvalid = (int)((R.B - in_launch < Geo<ROWS>::kChains) ? (R.B - in_launch) : Geo<ROWS>::kChains);
  if (nvalid < 0) nvalid = 0;   // (a pair's padding CTA)
  const uint32_t bytes = (uint32_t)(nvalid * d) * 4u;
  float* dst_tr = tr_now ? R.trace + (((R.t_call0 + t + 1) / R.thin - 1) * R.B_rows + first) * d : nullptr;
  float* dst_win = R.win ? R.win + (t * R.B_rows + first) * d : nullptr;
  const bool bulk = ((bytes | (uint32_t)reinterpret_cast<uintptr_t>(dst_tr) | (uint32_t)reinterpret_cast<uintptr_t>(dst_win)) & 15u) == 0u;
  if (bulk) {
    const uint32_t stage = C.sbase + SmemLayout::A + 49152u;
    if (valid) {
#pragma unroll
      for (int i = 0; i < 8; ++i)
        if (8 * C.k + i < d) ptx::sts_32(stage + (uint32_t)(C.row * d + 8 * C.k + i) * 4u, cur[i]);
    }
    ptx::named_bar_sync(9, Geo<ROWS>::kChains * 4);
    if (C.row == 0 && C.k == 0 && nvalid > 0) {
      ptx::fence_proxy_async();
      if (dst_tr) ptx::bulk_s2g(dst_tr, stage, bytes);
      if (dst_win) ptx::bulk_s2g(dst_win, stage, bytes);
      ptx::bulk_commit();
      C.emit_pending = 1;
    }
  } else if (valid) {
    const int64_t off = (int64_t)C.row * d + 8 * C.k;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (8 * C.k + i < d) {
        if (dst_tr) dst_tr[off + i] = cur[i];
        if (dst_win) dst_win[off + i] = cur[i];
      }
    }
  }
}

template <int METHOD, int ROWS>
__device__ __forceinline__ void sampler_thread(EpiCtx& C, const Run& R) {
  const Params& P = *C.P;
  const int d = P.d;
  if (METHOD == M_EVAL) {
    // tile loop (Run::n_tiles): both CTAs of a pair make the same number of passes (n_tiles and gridDim.x are even)
    for (int64_t tile = blockIdx.x; tile < R.n_tiles; tile += gridDim.x) {
      const int64_t r_in_launch = tile * Geo<ROWS>::kChains + C.row;
      const bool valid = r_in_launch < R.B;
      float th[8], g[8], lp;
      if (R.io_mode == IO_ROWS_F32) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int gi = 8 * C.k + i;
          th[i] = (valid && gi < d) ? R.in_rows[r_in_launch * d + gi] : 0.0f;
        }
      } else {
        load_vec8(C, R.theta, R.ld, r_in_launch, d, valid, th);
      }
      eval_target<ROWS>(C, th, R.want_grad != 0, lp, g);
      if (valid) {
        if (R.io_mode == IO_ROWS_F32) {
          if (C.k == 0) R.out_logp[r_in_launch] = lp;
          if (R.want_grad) {
#pragma unroll
            for (int i = 0; i < 8; ++i) if (8 * C.k + i < d) R.out_grad[r_in_launch * d + 8 * C.k + i] = g[i];
          }
        } else {
          if (C.k == 0) R.logp[r_in_launch] = (double)lp;
          if (R.want_grad) store_vec8(C, R.grad, R.ld, r_in_launch, d, g);
        }
      }
    }
    return;
  }

  const int64_t r_in_launch = (int64_t)blockIdx.x * Geo<ROWS>::kChains + C.row;
  const bool valid = r_in_launch < R.B;
  const bool lead = valid && C.k == 0;

  if (METHOD == M_AIES) {
    const int64_t i = R.own0 + r_in_launch;
    const uint32_t cid = R.chain0 + (uint32_t)i;
    const uint4 w = philox4x32_10(cid, R.step0, 0u, R.seed);
    const int64_t j = R.oth0 + (int64_t)__umulhi(w.z, (uint32_t)R.n_oth);
    const float a = R.eps;
    const float t = u01<float>(w.y) * (a - 1.0f) + 1.0f;
    const float z = t * t / a;
    float thp[8], thi[8], g[8], lpp;
    if (R.de) {
      // eq (2.16), reading R23: x' = x_i + gamma (x_j - x_k), k != j from the same half, R.eps = sigma_gamma
      int64_t kr = (int64_t)__umulhi(w.w, (uint32_t)(R.n_oth - 1));
      if (kr >= j - R.oth0) kr += 1;
      const uint4 wn = philox4x32_10(cid, R.step0, 1u, R.seed);
      float n0, n1;
      box_muller(wn.x, wn.y, n0, n1);
      const float gamma = (1.0f + R.eps * n0) * (2.38f / sqrtf(2.0f * (float)d));
      float thj[8], thk[8];
      load_vec8(C, R.theta, R.ld, i, d, valid, thi);
      load_vec8(C, R.theta, R.ld, j, d, valid, thj);
      load_vec8(C, R.theta, R.ld, R.oth0 + kr, d, valid, thk);
#pragma unroll
      for (int q = 0; q < 8; ++q) thp[q] = thi[q] + gamma * (thj[q] - thk[q]);
    } else {
      float thj[8];
      load_vec8(C, R.theta, R.ld, i, d, valid, thi);
      load_vec8(C, R.theta, R.ld, j, d, valid, thj);
#pragma unroll
      for (int q = 0; q < 8; ++q) thp[q] = thj[q] + z * (thi[q] - thj[q]);
    }
    eval_target<ROWS>(C, thp, false, lpp, g);
    const float la = (R.de ? 0.0f : (float)(d - 1) * logf(z)) + lpp - (valid ? (float)R.logp[i] : 0.0f);
    const bool acc = valid && accept_rule<float>(u01<float>(w.x), la);
    qbar(C);   // (warp-uniform) every thread of the chain has read logp[i] before the leader overwrites it
    if (acc) store_vec8(C, R.theta, R.ld, i, d, thp);
    if (lead) {
      R.last_la[i] = (double)la;
      if (acc) { R.logp[i] = (double)lpp; R.n_accept[i] += 1ull; }
    }
    if (R.trace) {   // every half-ensemble launch writes its own walkers (their state is final for this step)
      if (valid && !acc) load_vec8(C, R.theta, R.ld, i, d, valid, thp);
      emit_tile<ROWS>(C, R, 0, R.own0 + (int64_t)blockIdx.x * Geo<ROWS>::kChains, d, thp, valid);
      if (C.emit_pending) ptx::bulk_wait0();
    }
    return;
  }

  const int64_t c = r_in_launch;
  const uint32_t cid = R.chain0 + (uint32_t)c;
  const bool rows_out = (R.trace != nullptr) || (R.win != nullptr);
  const int64_t tile0 = (int64_t)blockIdx.x * Geo<ROWS>::kChains;   // first chain of this CTA's tile
  const float eps = R.eps;
  float lp = valid ? (float)R.logp[c] : 0.0f;
  float la_last = 0.0f;
  unsigned long long nacc = 0;

  if (METHOD == M_MH) {
    float th[8];
    load_vec8(C, R.theta, R.ld, c, d, valid, th);
    for (int64_t t = 0; t < R.n_steps; ++t) {
      const uint64_t step = R.step0 + (uint64_t)t;
      float thp[8], g[8], lpp;
      {
        float xi[8], dx[8];
        draw_normals8(C, R.seed, cid, step, d, xi);
#pragma unroll
        for (int i = 0; i < 8; ++i) xi[i] *= eps;
        mv_L(C, xi, dx);
#pragma unroll
        for (int i = 0; i < 8; ++i) thp[i] = th[i] + dx[i];
      }
      eval_target<ROWS>(C, thp, false, lpp, g);
      const float la = lpp - lp;
      la_last = la;
      const uint4 w = philox4x32_10(cid, step, 0u, R.seed);
      if (valid && accept_rule<float>(u01<float>(w.x), la)) {
#pragma unroll
        for (int i = 0; i < 8; ++i) th[i] = thp[i];
        lp = lpp;
        ++nacc;
      }
      if (rows_out) emit_tile<ROWS>(C, R, t, tile0, d, th, valid);
    }
    if (valid) store_vec8(C, R.theta, R.ld, c, d, th);
  }

  if (METHOD == M_MALA) {
    const float sq = sqrtf(2.0f * eps);
    // The whitened gradient L^T g of the current state stays in registers across the steps: the proposal's
    // L^T g' is needed for the Hastings ratio anyway and becomes it on acceptance (the same fp32 values the
    // matvec would reproduce from the stored gradient, so a call split into several gives the same bits).
    float gz[8];
    {
      float g[8];
      load_vec8(C, R.grad, R.ld, c, d, valid, g);
      mv_Lt(C, g, gz);
    }
    for (int64_t t = 0; t < R.n_steps; ++t) {
      const uint64_t step = R.step0 + (uint64_t)t;
      float thp[8], dz[8], gp[8], gzp[8], lpp, fwd = 0.0f;
      {
        float g[8], xi[8], th[8];
        load_vec8(C, R.theta, R.ld, c, d, valid, th);   // (requested before the normals are drawn)
        draw_normals8(C, R.seed, cid, step, d, xi);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float f = sq * xi[i];
          fwd = fmaf(f, f, fwd);
          dz[i] = fmaf(eps, gz[i], f);
        }
        mv_L(C, dz, g);  // g <- L dz
#pragma unroll
        for (int i = 0; i < 8; ++i) thp[i] = th[i] + g[i];
      }
      eval_target<ROWS>(C, thp, true, lpp, gp);
      float diff = fwd;
      mv_Lt(C, gp, gzp);
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float r = fmaf(eps, gzp[i], dz[i]);
        diff = fmaf(-r, r, diff);
      }
      const float la = lpp - lp + reduce4(C, diff) / (4.0f * eps);
      la_last = la;
      const uint4 w = philox4x32_10(cid, step, 0u, R.seed);
      const bool acc = valid && accept_rule<float>(u01<float>(w.x), la);
      if (acc) {
        store_vec8(C, R.theta, R.ld, c, d, thp);
        store_vec8(C, R.grad, R.ld, c, d, gp);
        lp = lpp;
        ++nacc;
#pragma unroll
        for (int i = 0; i < 8; ++i) gz[i] = gzp[i];
      }
      if (rows_out) {
        if (valid && !acc) load_vec8(C, R.theta, R.ld, c, d, valid, thp);
        emit_tile<ROWS>(C, R, t, tile0, d, thp, valid);
      }
    }
  }

  if (METHOD == M_HMC) {
    for (int64_t t = 0; t < R.n_steps; ++t) {
      const uint64_t step = R.step0 + (uint64_t)t;
      float thw[8], q[8], gw[8], lpw = lp, kin0 = 0.0f;
      {
        float g[8], gz[8];
        draw_normals8(C, R.seed, cid, step, d, q);
#pragma unroll
        for (int i = 0; i < 8; ++i) kin0 = fmaf(q[i], q[i], kin0);
        load_vec8(C, R.grad, R.ld, c, d, valid, g);
        mv_Lt(C, g, gz);
#pragma unroll
        for (int i = 0; i < 8; ++i) q[i] = fmaf(0.5f * eps, gz[i], q[i]);
        load_vec8(C, R.theta, R.ld, c, d, valid, thw);
      }
      for (int l = 1; l <= R.n_leapfrog; ++l) {
        {
          float dz[8], dx[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) dz[i] = eps * q[i];
          mv_L(C, dz, dx);
#pragma unroll
          for (int i = 0; i < 8; ++i) thw[i] += dx[i];
        }
        eval_target<ROWS>(C, thw, true, lpw, gw);
        float gz[8];
        mv_Lt(C, gw, gz);
        const float cc = (l < R.n_leapfrog) ? eps : 0.5f * eps;
#pragma unroll
        for (int i = 0; i < 8; ++i) q[i] = fmaf(cc, gz[i], q[i]);
      }
      float kin1 = 0.0f;
#pragma unroll
      for (int i = 0; i < 8; ++i) kin1 = fmaf(q[i], q[i], kin1);
      // log alpha = H0 - H1 = (lp' - lp) + (|q0|^2 - |q1|^2)/2
      const float la = (lpw - lp) + 0.5f * reduce4(C, kin0 - kin1);
      la_last = la;
      const uint4 w = philox4x32_10(cid, step, 0u, R.seed);
      const bool acc = valid && accept_rule<float>(u01<float>(w.x), la);
      if (acc) {
        store_vec8(C, R.theta, R.ld, c, d, thw);
        store_vec8(C, R.grad, R.ld, c, d, gw);
        lp = lpw;
        ++nacc;
      }
      if (rows_out) {
        if (valid && !acc) load_vec8(C, R.theta, R.ld, c, d, valid, thw);
        emit_tile<ROWS>(C, R, t, tile0, d, thw, valid);
      }
    }
  }

  if (lead) {
    R.logp[c] = (double)lp;
    R.last_la[c] = (double)la_last;
    R.n_accept[c] += nacc;
  }
  if (C.emit_pending) ptx::bulk_wait0();   // the staging area must outlive the copy
}

template <int METHOD, int ROWS>
__global__ void __launch_bounds__(kThreads, 1)
best_tc_kernel(const __grid_constant__ Params P, const __grid_constant__ Run R) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const int tid = threadIdx.x, lane = tid & 31;
  // the warp index through a shuffle: the compiler then knows the role branches are warp-uniform and keeps the MMA
  // issuer's descriptors, counters and barrier addresses in uniform registers
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const uint32_t sbase = ptx::smem_u32(smem);
  const Bars bars = make_bars(sbase + SmemLayout::BARS);
  float* bias_s = reinterpret_cast<float*>(smem + SmemLayout::BIAS);
  float* wouts_s = reinterpret_cast<float*>(smem + SmemLayout::WOUTS);
  float* Ls = reinterpret_cast<float*>(smem + SmemLayout::LMAT);
  float* LTs = reinterpret_cast<float*>(smem + SmemLayout::LTMAT);
  float* Rs = reinterpret_cast<float*>(smem + SmemLayout::RMAT);
  float* RTs = reinterpret_cast<float*>(smem + SmemLayout::RTMAT);
  float* vecs = reinterpret_cast<float*>(smem + SmemLayout::VECS);
  volatile uint32_t* tmem_ptr = reinterpret_cast<volatile uint32_t*>(smem + SmemLayout::TMEMPTR);

  if (tid == 0) {
    for (int i = 0; i < 8; ++i) {
      ptx::mbar_init(bars.full(i), 1); ptx::mbar_init(bars.empty(i), 1);
    }
    for (int i = 0; i < kMaxKch; ++i) {
      // arrivals per phase: in place = every epilogue thread (pair: the 256 of the lane half that owns the
      // k-chunk); L2-image tiles = warp 3 alone (+ the bulk copy's bytes)
      ptx::mbar_init(bars.a_ready(i), (!Geo<ROWS>::kInPlace) ? 1 : (Geo<ROWS>::kWide ? 2 : 1) * Geo<ROWS>::kEpiArrive);   // pair: half of each CTA's; 256: both CTAs'
      ptx::mbar_init(bars.a_free(i), Geo<ROWS>::kCluster ? 2 : 1);   // pair kernels: two issuing warps
    }
    for (int i = 0; i < 4; ++i) {
      ptx::mbar_init(bars.d_full(i), 1);
      ptx::mbar_init(bars.d_free(i), Geo<ROWS>::kCluster ? 2 * Geo<ROWS>::kEpiArrive : Geo<ROWS>::kEpiActive);   // pair: both CTAs
    }
    for (int i = 0; i < 4; ++i) ptx::mbar_init(bars.epi_done(i), Geo<ROWS>::kEpiActive);
    ptx::mbar_init(bars.xin_done(), Geo<ROWS>::kEpiActive);
    ptx::fence_mbar_init();
  }
  if (warp == 2) {
    if (Geo<ROWS>::kCluster) ptx::tmem_alloc_2cta(sbase + SmemLayout::TMEMPTR, 512);
    else ptx::tmem_alloc(sbase + SmemLayout::TMEMPTR, 512);
  }
  // Prologue tables.  Every global load is issued before the first shared-memory store, so that the tables cost one
  // memory round trip (they are cold after an L2 flush) instead of one per table.  The tables were 4-6 us of a launch
  // with the four loops one after the other (measured by skipping them), 2 us less this way: nothing for a 100-step
  // sampler call, 3-5 % of a one-pass best_logp_grad (16 384 points forward: 37.9 -> 35.8 us, with gradient 60.3 -> 58.4).
  {
    const int nb = P.bias16 ? (P.n_hidden * P.H) >> 1 : P.n_hidden * P.H;   // table words: <= 2048 (SmemLayout::BIAS)
    float2 bq[4];
    float wq[2];
    double lq[2], rq[2], m3[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = tid + u * kThreads;
      bq[u] = make_float2(0.0f, 0.0f);
      if (i < nb) {
        if (P.bias16) bq[u] = *reinterpret_cast<const float2*>(P.bias + 2 * i);
        else bq[u].x = P.bias[i];
      }
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int i = tid + u * kThreads;
      wq[u] = (i < P.H) ? P.w_out[i] : 0.0f;
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int i = tid + u * kThreads, r = i / kDP, c = i % kDP;
      lq[u] = (i < kDP * kDP && r < P.d && c <= r) ? P.L[r * P.d + c] : 0.0;
      rq[u] = (i < kDP * kDP && P.has_gauss && r < P.d && c < P.d && c >= r) ? P.R[r * P.d + c] : 0.0;
    }
    if (tid < P.d && tid < kDP) {
      if (P.has_gauss) m3[0] = P.mu[tid];
      if (P.has_box) { m3[1] = P.lo[tid]; m3[2] = P.hi[tid]; }
    }
    uint32_t* b16 = reinterpret_cast<uint32_t*>(bias_s);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = tid + u * kThreads;
      if (i < nb) {
        if (P.bias16) b16[i] = ptx::pack_bf16x2(bq[u].x, bq[u].y);   // bf16 bias table, two per word
        else bias_s[i] = bq[u].x;
      }
    }
    for (int i = tid + 4 * kThreads; i < nb; i += kThreads) {   // (not reached by the supported shapes)
      if (P.bias16) b16[i] = ptx::pack_bf16x2(P.bias[2 * i], P.bias[2 * i + 1]);
      else bias_s[i] = P.bias[i];
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int i = tid + u * kThreads;
      if (i < P.H) wouts_s[i] = 0.5f * (P.mlp_scale * wq[u]);   // see fwd_group (LAST)
    }
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int i = tid + u * kThreads, r = i / kDP, c = i % kDP;
      if (i < kDP * kDP) {
        const float l = (float)lq[u], uu = (float)rq[u];
        Ls[i] = l;
        LTs[c * kDP + r] = l;
        Rs[i] = uu;
        RTs[c * kDP + r] = uu;
      }
    }
    if (tid < kDP) {
      const bool in = tid < P.d;
      vecs[tid] = (in && P.has_gauss) ? (float)m3[0] : 0.0f;
      vecs[32 + tid] = (in && P.has_box) ? (float)m3[1] : -3.0e38f;
      vecs[64 + tid] = (in && P.has_box) ? (float)m3[2] : 3.0e38f;
      vecs[96 + tid] = (in && P.has_box) ? (float)(1.0 / (m3[2] - m3[1])) : 0.0f;
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  if (Geo<ROWS>::kCluster) ptx::cluster_sync_all();   // both CTAs' barriers initialised, both TMEM allocations made
  const uint32_t tmem_base = *tmem_ptr;

  int64_t n_evals = 1;
  if (METHOD == M_EVAL) n_evals = (R.n_tiles - (int64_t)blockIdx.x + (int64_t)gridDim.x - 1) / (int64_t)gridDim.x;
  if (METHOD == M_MH || METHOD == M_MALA) n_evals = R.n_steps;
  if (METHOD == M_HMC) n_evals = R.n_steps * R.n_leapfrog;
  const int n_ops = R.want_grad ? P.n_ops_all : P.n_ops_fwd;

  if (warp < kCtrlWarps) {
    if (Geo<ROWS>::kCluster) {
      const uint32_t rank = ptx::cluster_ctarank();
      if (warp == 0) {
        producer_loop_pair<ROWS>(P, bars, sbase + Geo<ROWS>::kStagesOff, rank, n_evals, n_ops);
      } else if ((warp == 1 || warp == 3) && rank == 0) {
        mma_loop_pair<true, ROWS>(P, bars, sbase + SmemLayout::A, sbase + Geo<ROWS>::kStagesOff, tmem_base, n_evals, n_ops,
                                  warp == 3 ? 1 : 0);
      }
    } else if (warp == 0) {
      producer_loop(P, bars, sbase + SmemLayout::STAGES, n_evals, n_ops);
    } else if (warp == 1) {
      mma_loop<ROWS>(P, bars, sbase + SmemLayout::A, sbase + SmemLayout::STAGES, tmem_base, n_evals, n_ops);
    } else if ((!Geo<ROWS>::kInPlace) && warp == 3) {
      loader_loop(P, bars, sbase + SmemLayout::A, P.aimg + (size_t)blockIdx.x * (16u * Geo<ROWS>::kAChunk),
                  Geo<ROWS>::kAChunk, n_evals, n_ops);
    }
  } else {
    EpiCtx C;
    C.P = &P;
    C.bars = bars;
    C.sbase = sbase;
    C.row = Geo<ROWS>::kPair ? ((warp & 1) * 32 + lane) : ((warp & 3) * 32 + lane);
    C.half = Geo<ROWS>::kPair ? ((warp & 3) >> 1) : 0;
    C.to_leader = (Geo<ROWS>::kCluster && ptx::cluster_ctarank() != 0) ? 1 : 0;
    C.k = (warp - kCtrlWarps) >> 2;
    C.tmem_lane = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
    C.o = 0; C.g = 0; C.vslot = 0; C.pslot = 0; C.emit_pending = 0;
    if (Geo<ROWS>::kOwn) {   // chunk-owner epilogue: bases without the k offsets (store_piece, fwd_group colofs)
      C.a_thr0 = sbase + SmemLayout::A + C.row * 128;
      C.a_thr1 = (uint32_t)(C.row & 7);
      C.bias_thr = sbase + SmemLayout::BIAS;
      C.wouts_thr = sbase + SmemLayout::WOUTS;
      C.dact_thr = reinterpret_cast<uint8_t*>(P.dact + (size_t)blockIdx.x * P.dact_tile_elems) + (size_t)C.row * 16u;
    } else {
      C.a_thr0 = sbase + SmemLayout::A + C.row * 128 + (((2 * C.k) ^ (C.row & 7)) << 4);
      C.a_thr1 = sbase + SmemLayout::A + C.row * 128 + (((2 * C.k + 1) ^ (C.row & 7)) << 4);
      C.bias_thr = sbase + SmemLayout::BIAS + C.k * (P.bias16 ? 32 : 64);
      C.wouts_thr = sbase + SmemLayout::WOUTS + C.k * 64;
      C.dact_thr = reinterpret_cast<uint8_t*>(P.dact + (size_t)blockIdx.x * P.dact_tile_elems) +
                   (size_t)(2 * C.k * Geo<ROWS>::kTileRows + C.row) * 16u;
    }
    C.v_thr = (uint32_t)C.row * 8u;
    C.aimg_thr = (!Geo<ROWS>::kInPlace) ? P.aimg + (size_t)blockIdx.x * (16u * Geo<ROWS>::kAChunk) + C.row * 128 + (((2 * C.k) ^ (C.row & 7)) << 4)
                     : nullptr;
    if (C.row >= Geo<ROWS>::kChains) {
      // phantom rows (geometry 233: the odd row quarters; L2-image tiles: lanes ROWS..127): nothing to do
    } else if (Geo<ROWS>::kPair && C.half == 1) {
      // upper lane half of a CTA pair: MLP epilogues only, in step with the sampler threads
      const float th0[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      float gm[8], op_;
      for (int64_t e = 0; e < n_evals; ++e) tc_eval<ROWS>(C, th0, R.want_grad != 0, op_, gm);
    } else {
      sampler_thread<METHOD, ROWS>(C, R);
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (Geo<ROWS>::kCluster) ptx::cluster_sync_all();   // the leader's MMAs wrote the peer's TMEM and read its SMEM
  if (warp == 2) {
    if (Geo<ROWS>::kCluster) ptx::tmem_dealloc_2cta(tmem_base, 512);
    else ptx::tmem_dealloc(tmem_base, 512);
  }
}

}  // namespace tc

// =================================================================================================
// host side
// =================================================================================================
struct TcPlan {
  tc::Params P{};
  tc::Params Pp{};           // 512-wide ping-pong pairs (geometry 265): the same ops in the paired order, own weight pack
  bool has_pp = false;
  uint8_t* wpack = nullptr;
  uint8_t* wpack_p = nullptr;
  tc::Params Pn{};           // geometry 233: N-chunk outer order with the permuted row blocks, own weight pack
  uint8_t* wpack_n = nullptr;
  float* bias = nullptr;
  float* w_out = nullptr;
  uint16_t* dact = nullptr;
  uint8_t* aimg = nullptr;
  size_t dact_cap = 0, aimg_cap = 0;
  int n_sm = 0;
  int force_rows = 0;   // BEST_TC_ROWS (environment, read at best_create; documented in best.h): tests force a geometry
};

namespace {

uint16_t f32_to_bf16(float f) {  // round to nearest even
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((u >> 16) | 0x40);
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

template <int METHOD, int ROWS>
int launch_tc_geo(best_ctx* ctx, const tc::Run& R, int64_t rows, cudaStream_t s) {
  TcPlan* pl = ctx->tc;
  tc::Params& P = (ROWS == 265 && pl->has_pp) ? pl->Pp
                : (ROWS == 233 && pl->has_pp) ? pl->Pn : pl->P;
  constexpr int kTileRows = tc::Geo<ROWS>::kTileRows, kChains = tc::Geo<ROWS>::kChains;
  int64_t n_tiles = (rows + kChains - 1) / kChains;
  if (tc::Geo<ROWS>::kCluster) n_tiles = (n_tiles + 1) & ~(int64_t)1;   // whole CTA pairs
  // scratch: act' blocks (forward -> backward) and, for ROWS < 128, the next-operand image
  P.dact_tile_elems = (size_t)(P.n_hidden - 1) * P.H * kTileRows;
  const size_t dact_bytes = sizeof(uint16_t) * P.dact_tile_elems * (size_t)n_tiles + 16;
  const size_t aimg_bytes = tc::Geo<ROWS>::kInPlace ? 16 : (size_t)16 * tc::Geo<ROWS>::kAChunk * (size_t)n_tiles;
  if (dact_bytes > pl->dact_cap || aimg_bytes > pl->aimg_cap) {
    BEST_CUDA(cudaStreamSynchronize(s));
    if (dact_bytes > pl->dact_cap) {
      if (pl->dact) cudaFree(pl->dact);
      pl->dact = nullptr; pl->dact_cap = 0;
      BEST_CUDA(cudaMalloc(&pl->dact, dact_bytes));
      pl->dact_cap = dact_bytes;
    }
    if (aimg_bytes > pl->aimg_cap) {
      if (pl->aimg) cudaFree(pl->aimg);
      pl->aimg = nullptr; pl->aimg_cap = 0;
      BEST_CUDA(cudaMalloc(&pl->aimg, aimg_bytes));
      pl->aimg_cap = aimg_bytes;
    }
  }
  P.dact = pl->dact;
  P.aimg = pl->aimg;
  static std::atomic<bool> attr_set{false};   // idempotent: a race only repeats the call
  const int smem_bytes = tc::SmemLayout::TOTAL + 1024;
  if (!attr_set.load(std::memory_order_acquire)) {
    BEST_CUDA(cudaFuncSetAttribute(tc::best_tc_kernel<METHOD, ROWS>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    attr_set.store(true, std::memory_order_release);
  }
  P.L = ctx->L_dev;
  P.hard_box = ctx->tgt.hard_box;
  tc::Run Rl = R;
  int64_t grid = n_tiles;
  if (METHOD == tc::M_EVAL) {
    // best_logp_grad / cache refresh: one wave of CTAs walks all tiles (Run::n_tiles).  The wave is what the device
    // holds at once: CTA pairs cannot straddle GPCs, so ask the occupancy calculator instead of assuming n_sm / 2.
    static std::atomic<int> wave{0};
    int w = wave.load(std::memory_order_acquire);
    if (w == 0) {
      if (tc::Geo<ROWS>::kCluster) {
        cudaLaunchConfig_t q{};
        q.gridDim = dim3(2 * (unsigned)pl->n_sm); q.blockDim = dim3(tc::kThreads); q.dynamicSmemBytes = (size_t)smem_bytes;
        cudaLaunchAttribute qa[1];
        qa[0].id = cudaLaunchAttributeClusterDimension;
        qa[0].val.clusterDim.x = 2; qa[0].val.clusterDim.y = 1; qa[0].val.clusterDim.z = 1;
        q.attrs = qa; q.numAttrs = 1;
        int nc = 0;
        BEST_CUDA(cudaOccupancyMaxActiveClusters(&nc, tc::best_tc_kernel<METHOD, ROWS>, &q));
        w = 2 * nc;
      } else {
        int nb = 0;
        BEST_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, tc::best_tc_kernel<METHOD, ROWS>, tc::kThreads, (size_t)smem_bytes));
        w = nb * pl->n_sm;
      }
      if (w < 2) w = 2;
      wave.store(w, std::memory_order_release);
    }
    Rl.n_tiles = n_tiles;
    if (grid > w) grid = w;
  }
  if (tc::Geo<ROWS>::kCluster) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(tc::kThreads);
    cfg.dynamicSmemBytes = (size_t)smem_bytes;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    BEST_CUDA(cudaLaunchKernelEx(&cfg, tc::best_tc_kernel<METHOD, ROWS>, P, Rl));
  } else {
    tc::best_tc_kernel<METHOD, ROWS><<<(unsigned)grid, tc::kThreads, smem_bytes, s>>>(P, Rl);
  }
  count_launch();
  BEST_CUDA(cudaGetLastError());
  return BEST_OK;
}

// Chains per CTA.  Measured on B200 (27->512^4->1, one CTA alone, HMC ms per 128 evaluations):
// 128-chain in-place tiles 6.69, 64-chain 9.33, 32-chain 7.82 -- the L2 round trip of the operand
// costs more than the smaller epilogue saves, so widths <= 512 always use 128-chain tiles; only
// 1024-wide layers (whose operand does not fit in place) use 64, or 32 when that fills more SMs.
int pick_rows(const TcPlan* pl, int64_t rows, int n_sm) {
  if (pl->force_rows) return pl->force_rows;
  if (pl->P.H == 512) {
    // 512-wide: 128-chain single-CTA tiles or 64-chain CTA pairs (operand + accumulators double-buffered).
    // Measured per evaluation of one tile (HMC, B200): 52 us against 33 us, so the pairs win whenever
    // they do not need more waves of CTAs: the 4096-chain config, the small points of the sweep.
    // Geometry 233 (32 chains per CTA of a pair, the other 32 MMA rows phantom) has the same tensor work per
    // CTA as 265 and half the epilogue work: measured 36.1 us against 38.7 us per MALA step of a tile, so it
    // wins only while twice the CTAs still fit in one wave (4096 chains: 128 CTAs on 148 SMs, +7 %).
    const int64_t t128 = (rows + 127) / 128, t64 = ((rows + 63) / 64 + 1) & ~(int64_t)1,
                  t32 = ((rows + 31) / 32 + 1) & ~(int64_t)1;
    const int64_t pair_slots = n_sm & ~1;   // CTAs of whole pairs resident at once
    const double c128 = (double)((t128 + n_sm - 1) / n_sm) * 52.0, c265 = (double)((t64 + pair_slots - 1) / pair_slots) * 33.0,
                 c233 = (double)((t32 + pair_slots - 1) / pair_slots) * 30.8;
    // Geometry 256 (128-chain tiles on CTA pairs: half the shared-memory operand traffic of the MMAs per SM)
    // measured against 128 on 16 384 chains: HMC 6.32 -> 5.61 ms per launch, MALA 5.67 -> 4.97, MH 2.44 -> 2.39.
    const int64_t t256 = (t128 + 1) & ~(int64_t)1;
    const double c256 = (double)((t256 + pair_slots - 1) / pair_slots) * 46.0;
    if (c233 < c265 && c233 < c128 && c233 < c256) return 233;
    if (c265 < c128 && c265 < c256) return 265;
    return c256 <= c128 ? 256 : 128;
  }
  if (pl->P.H != 1024) return 128;
  // CTA pairs (cta_group::2): the 1024-wide operand in place at full MMA rate; 32 chains per CTA (geometry 232)
  // while twice the CTAs still fit one wave, as 233 for 512-wide layers
  const int64_t t32 = ((rows + 31) / 32 + 1) & ~(int64_t)1;
  return t32 <= (n_sm & ~1) ? 232 : 264;
}

template <int METHOD>
int launch_tc(best_ctx* ctx, const tc::Run& R, int64_t rows, cudaStream_t s) {
  TcPlan* pl = ctx->tc;
  if (pl->n_sm == 0) {
    int dev = 0;
    BEST_CUDA(cudaGetDevice(&dev));
    BEST_CUDA(cudaDeviceGetAttribute(&pl->n_sm, cudaDevAttrMultiProcessorCount, dev));
  }
  switch (pick_rows(pl, rows, pl->n_sm)) {
    case 128: return launch_tc_geo<METHOD, 128>(ctx, R, rows, s);
    case 256: return launch_tc_geo<METHOD, 256>(ctx, R, rows, s);
    case 264: return launch_tc_geo<METHOD, 264>(ctx, R, rows, s);
    case 265: return launch_tc_geo<METHOD, 265>(ctx, R, rows, s);
    case 233: return launch_tc_geo<METHOD, 233>(ctx, R, rows, s);
    case 232: return launch_tc_geo<METHOD, 232>(ctx, R, rows, s);
    case 64: return launch_tc_geo<METHOD, 64>(ctx, R, rows, s);
    default: return launch_tc_geo<METHOD, 32>(ctx, R, rows, s);
  }
}

}  // namespace

// the weight pack as a 2-D byte tensor for the CTA-pair kernel's 2-SM tensor copies
static int make_wmap(CUtensorMap* m, void* base, size_t bytes, uint32_t box_rows) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn enc = nullptr;
  if (!enc) {
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult qr;
    BEST_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qr));
    if (!fp || qr != cudaDriverEntryPointSuccess) { set_error("cuTensorMapEncodeTiled not available"); return BEST_ERR_CUDA; }
    enc = (encode_fn)fp;
  }
  const cuuint64_t dims[2] = {256, (cuuint64_t)(bytes / 256)};   // box dimensions are limited to 256 elements
  const cuuint64_t strides[1] = {256};
  const cuuint32_t box[2] = {256, box_rows};
  const cuuint32_t es[2] = {1, 1};
  const CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { set_error("cuTensorMapEncodeTiled failed"); return BEST_ERR_CUDA; }
  return BEST_OK;
}

int tc_plan_create(best_ctx* ctx, const best_config* cfg) {
  const int K = cfg->n_affine - 1;  // hidden layers
  if (K < 1) { set_error("BEST_PREC_BF16 needs at least one hidden layer"); return BEST_ERR_UNSUPPORTED; }
  const int H = cfg->widths[1];
  for (int k = 1; k <= K; ++k)
    if (cfg->widths[k] != H) { set_error("BEST_PREC_BF16: hidden widths must be equal"); return BEST_ERR_UNSUPPORTED; }
  const bool r64 = (H == 1024);
  if (!(H == 64 || H == 128 || H == 256 || H == 512 || H == 1024) || K * H > (r64 ? 4096 : 2048) ||
      2 * K > tc::kMaxOps) {
    set_error("BEST_PREC_BF16: hidden width must be 64/128/256/512 (n_hidden*width <= 2048) or 1024 (<= 4096)");
    return BEST_ERR_UNSUPPORTED;
  }
  const int d = cfg->d;
  TcPlan* pl = new TcPlan();
  ctx->tc = pl;
  if (const char* e = std::getenv("BEST_TC_ROWS")) {
    const int v = std::atoi(e);
    if ((v == 64 || v == 32 || (v == 128 && !r64) || ((v == 264 || v == 232) && r64) || ((v == 265 || v == 233 || v == 256) && H == 512))) pl->force_rows = v;
  }
  tc::Params& P = pl->P;
  P.bias16 = r64 ? 1 : 0;
  P.kch_max = H / 64;
  P.d = d; P.H = H; P.n_hidden = K; P.act = cfg->activation; P.mlp_scale = cfg->mlp_scale;
  const int ncols = H < 256 ? H : 256, nch = H / ncols, kchH = H / 64;
  // 1024-wide layers on the CTA-pair kernel: N-chunks issued two at a time (not for the forced fallbacks)
  const int paired = (r64 && pl->force_rows != 64 && pl->force_rows != 32) ? 1 : 0;
  int no = 0;
  for (int l = 0; l < K; ++l)
    P.ops[no++] = tc::OpDesc{l == 0 ? 1 : kchH, nch, ncols, l == K - 1 ? tc::EPI_FWD_LAST : tc::EPI_FWD_HID, l, paired, paired};
  P.n_ops_fwd = no;
  for (int l = K - 1; l >= 1; --l) P.ops[no++] = tc::OpDesc{kchH, nch, ncols, tc::EPI_BWD_HID, l - 1, paired, paired};
  P.ops[no++] = tc::OpDesc{kchH, 1, 32, tc::EPI_BWD_FINAL, 0, 0};
  P.n_ops_all = no;
  P.dact_tile_elems = 0;   // set per launch (depends on the tile geometry)

  // host views of the fp32 weights
  std::vector<const float*> W(K + 1);
  std::vector<const float*> bvec(K + 1);
  {
    size_t wo = 0, bo = 0;
    for (int k = 0; k <= K; ++k) {
      W[k] = cfg->W_flat + wo;
      bvec[k] = cfg->b_flat + bo;
      wo += (size_t)cfg->widths[k] * cfg->widths[k + 1];
      bo += cfg->widths[k + 1];
    }
  }
  // B operand of every op as a logical [N][Ktot] bf16 matrix, cut into pre-swizzled stage tiles
  auto build_pack = [&](const tc::Params& PP) {
  std::vector<uint16_t> pack;
  for (int oi = 0; oi < PP.n_ops_all; ++oi) {
    const tc::OpDesc op = PP.ops[oi];
    // forward SiLU layers are packed pre-scaled by 1/2 (exact), see silu_pair()
    const float fs = (tc::kSiluHalfPrescale && cfg->activation == BEST_ACT_SILU) ? 0.5f : 1.0f;
    auto Bm = [&](int n, int k) -> float {
      if (op.epi == tc::EPI_FWD_HID || op.epi == tc::EPI_FWD_LAST) {
        if (op.layer == 0) { const int kk = k & 31; return kk < d ? fs * W[0][(size_t)n * d + kk] : 0.0f; }
        return fs * W[op.layer][(size_t)n * H + k];
      }
      if (op.epi == tc::EPI_BWD_HID) return 0.5f * W[op.layer + 1][(size_t)k * H + n];  // (W_l)^T / 2, l = layer+1 (silu_pair)
      return n < d ? W[0][(size_t)k * d + n] : 0.0f;                             // (W_0)^T
    };
    // consumption order of the K32 tiles: N-chunk outer, or (paired ops) two N-chunks at a time with the
    // 64-wide k-chunk outer
    std::vector<std::pair<int, int>> order;   // (c, k32)
    if (op.paired) {
      for (int c = 0; c < op.nch; c += 2)
        for (int j = 0; j < op.kch; ++j)
          for (int q = 0; q < 2; ++q) { order.push_back({c + q, 2 * j}); order.push_back({c + q, 2 * j + 1}); }
    } else {
      for (int c = 0; c < op.nch; ++c)
        for (int k32 = 0; k32 < 2 * op.kch; ++k32) order.push_back({c, k32});
    }
    for (const auto& ck : order) {
      const int c = ck.first, k32 = ck.second;
      {
        const size_t base = pack.size();
        pack.resize(base + (size_t)op.ncols * 32, 0);
        for (int r = 0; r < op.ncols; ++r)
          for (int kk = 0; kk < 32; ++kk) {
            const size_t off = (size_t)r * 32 + ((((kk >> 3) ^ ((r >> 1) & 3))) << 3) + (kk & 7);
            // paired ops (CTA-pair kernels): B row blocks in the order 0,2,1,3, see pair_jn()
            const int rl = (op.perm && op.ncols == 256) ? ((((r >> 6) & 1) * 2 + (r >> 7)) << 6) + (r & 63) : r;
            const float wv = Bm(c * op.ncols + rl, k32 * 32 + kk);
            pack[base + off] = f32_to_bf16(wv);
          }
      }
    }
  }
  pack.resize((pack.size() + 8191) / 8192 * 8192 + 8192, 0);   // whole 1 KB rows (+ slack) for the tensor maps
  return pack;
  };
  const std::vector<uint16_t> pack = build_pack(P);
  std::vector<float> bias((size_t)K * H);
  {
    const float fs = (tc::kSiluHalfPrescale && cfg->activation == BEST_ACT_SILU) ? 0.5f : 1.0f;
    for (int l = 0; l < K; ++l)
      for (int i = 0; i < H; ++i) bias[(size_t)l * H + i] = fs * bvec[l][i];
  }
  P.b_out = bvec[K][0];
  int rc;
  if ((rc = dev_alloc(&pl->wpack, pack.size() * 2))) return rc;
  if ((rc = dev_alloc(&pl->bias, bias.size()))) return rc;
  if ((rc = dev_alloc(&pl->w_out, (size_t)H))) return rc;
  BEST_CUDA(cudaMemcpy(pl->wpack, pack.data(), pack.size() * 2, cudaMemcpyHostToDevice));
  BEST_CUDA(cudaMemcpy(pl->bias, bias.data(), bias.size() * 4, cudaMemcpyHostToDevice));
  BEST_CUDA(cudaMemcpy(pl->w_out, W[K], sizeof(float) * H, cudaMemcpyHostToDevice));
  P.wpack = pl->wpack; P.bias = pl->bias; P.w_out = pl->w_out;
  if (r64 || H == 512) {
    if ((rc = make_wmap(&P.wmap8, pl->wpack, pack.size() * 2, 32))) return rc;
    if ((rc = make_wmap(&P.wmap1, pl->wpack, pack.size() * 2, 4))) return rc;
  }
  P.has_gauss = ctx->tgt.has_gauss; P.has_box = ctx->tgt.has_box;
  P.banana_i = ctx->tgt.banana_i; P.banana_j = ctx->tgt.banana_j;
  P.banana_sigma = (float)ctx->tgt.banana_sigma;
  P.pen_kappa = (float)ctx->tgt.pen_kappa; P.pen_gamma = (float)ctx->tgt.pen_gamma;
  P.mu = ctx->tgt.mu; P.R = ctx->tgt.R; P.lo = ctx->tgt.lo; P.hi = ctx->tgt.hi; P.L = ctx->L_dev;
  if (H == 512) {
    // geometry 265 issues the two N-chunks of a layer from two warps (k-chunk outer): same ops, paired order
    pl->Pp = P;
    for (int oi = 0; oi + 1 < P.n_ops_all; ++oi) pl->Pp.ops[oi].paired = pl->Pp.ops[oi].perm = 1;
    const std::vector<uint16_t> pack_p = build_pack(pl->Pp);
    if ((rc = dev_alloc(&pl->wpack_p, pack_p.size() * 2))) return rc;
    BEST_CUDA(cudaMemcpy(pl->wpack_p, pack_p.data(), pack_p.size() * 2, cudaMemcpyHostToDevice));
    pl->Pp.wpack = pl->wpack_p;
    if ((rc = make_wmap(&pl->Pp.wmap8, pl->wpack_p, pack_p.size() * 2, 32))) return rc;
    if ((rc = make_wmap(&pl->Pp.wmap1, pl->wpack_p, pack_p.size() * 2, 4))) return rc;
    pl->has_pp = true;
    // geometry 233: N-chunk outer (one issuing warp; the epilogue of the first N-chunk overlaps the MMAs of
    // the second) with the permuted row blocks, own pack.
    pl->Pn = P;
    for (int oi = 0; oi + 1 < P.n_ops_all; ++oi) pl->Pn.ops[oi].perm = 1;
    const std::vector<uint16_t> pack_n = build_pack(pl->Pn);
    if ((rc = dev_alloc(&pl->wpack_n, pack_n.size() * 2))) return rc;
    BEST_CUDA(cudaMemcpy(pl->wpack_n, pack_n.data(), pack_n.size() * 2, cudaMemcpyHostToDevice));
    pl->Pn.wpack = pl->wpack_n;
    if ((rc = make_wmap(&pl->Pn.wmap8, pl->wpack_n, pack_n.size() * 2, 32))) return rc;
    if ((rc = make_wmap(&pl->Pn.wmap1, pl->wpack_n, pack_n.size() * 2, 4))) return rc;
  }
  return BEST_OK;
}

void tc_plan_destroy(best_ctx* ctx) {
  TcPlan* pl = ctx->tc;
  if (!pl) return;
  cudaFree(pl->wpack); cudaFree(pl->wpack_p); cudaFree(pl->wpack_n); cudaFree(pl->bias); cudaFree(pl->w_out); cudaFree(pl->dact); cudaFree(pl->aimg);
  delete pl;
  ctx->tc = nullptr;
}

int tc_logp_grad(best_ctx* ctx, const float* theta_rows, int64_t n, float* logp, float* grad, cudaStream_t s) {
  tc::Run R{};
  R.method = tc::M_EVAL; R.want_grad = grad ? 1 : 0; R.io_mode = tc::IO_ROWS_F32;
  R.B = n; R.ld = n; R.n_steps = 1;
  R.in_rows = theta_rows; R.out_logp = logp; R.out_grad = grad;
  return launch_tc<tc::M_EVAL>(ctx, R, n, s);
}

// log pi and gradient at the state's theta into logp_out / grad_out (SoA fp64 [d][B]); the caller decides
// whether these are the state's caches
int tc_eval_state(best_ctx* ctx, best_state* st, double* logp_out, double* grad_out, cudaStream_t s) {
  tc::Run R{};
  R.method = tc::M_EVAL; R.want_grad = 1; R.io_mode = tc::IO_SOA_F64;
  R.B = st->B; R.ld = st->B; R.n_steps = 1;
  R.theta = st->theta; R.grad = grad_out; R.logp = logp_out;
  BEST_TRY(launch_tc<tc::M_EVAL>(ctx, R, st->B, s));
  st->n_evals += (uint64_t)st->B;
  return BEST_OK;
}

int tc_state_init(best_ctx* ctx, best_state* st, cudaStream_t s) {
  BEST_TRY(tc_eval_state(ctx, st, st->logp, st->grad, s));
  st->grad_valid = true;
  return BEST_OK;
}

// One best_step_* call = ONE persistent launch (two per step for the ensemble moves: the half-ensembles
// depend on each other device-wide).  The kernel writes the trace slots itself.  Under covariance adaptation
// (A9) the call is cut only where it must be: at a window boundary (the whitening factor changes there and
// every CTA reads it at launch) and when the window buffer -- fp32 rows of every post-accept state, written by
// the kernel -- is full; after each segment ONE Gram kernel folds the buffer into the fp64 window sums.
int tc_step(best_ctx* ctx, best_state* st, int method, int64_t n_steps, uint64_t seed, float eps,
            int n_leapfrog, float* trace, int thin, cudaStream_t s, bool de) {
  if ((method == tc::M_MALA || method == tc::M_HMC) && !st->grad_valid) BEST_TRY(tc_state_init(ctx, st, s));
  tc::Run R{};
  R.method = method; R.io_mode = tc::IO_SOA_F64;
  R.want_grad = (method == tc::M_MALA || method == tc::M_HMC) ? 1 : 0;
  R.B = st->B; R.ld = st->B; R.seed = seed; R.eps = eps; R.n_leapfrog = n_leapfrog;
  R.de = de ? 1 : 0;
  R.chain0 = (uint32_t)st->chain0;
  R.theta = st->theta; R.grad = st->grad; R.logp = st->logp; R.last_la = st->last_la; R.n_accept = st->n_accept;
  R.B_rows = st->B;
  if (trace && thin > 0) { R.trace = trace; R.thin = thin; } else { R.trace = nullptr; R.thin = 1; }
  const bool adapt = st->adapt_every > 0 && method != tc::M_AIES;
  int64_t t0 = 0;
  while (t0 < n_steps) {
    int64_t seg = n_steps - t0;
    if (adapt) {
      seg = std::min<int64_t>(seg, st->adapt_every - st->win_steps);
      seg = std::min<int64_t>(seg, st->win_cap_steps);
    }
    if (method == tc::M_AIES) seg = 1;
    R.n_steps = seg;
    R.step0 = st->step + (uint64_t)t0;
    R.t_call0 = t0;
    int wb = 0;
    if (adapt) BEST_TRY(adapt_acquire_buffer(st, s, &wb));
    R.win = adapt ? st->win_buf[wb] : nullptr;
    switch (method) {
      case tc::M_MH: BEST_TRY(launch_tc<tc::M_MH>(ctx, R, st->B, s)); break;
      case tc::M_MALA: BEST_TRY(launch_tc<tc::M_MALA>(ctx, R, st->B, s)); break;
      case tc::M_HMC: BEST_TRY(launch_tc<tc::M_HMC>(ctx, R, st->B, s)); break;
      default: {
        const int64_t half = st->B / 2;
        // sharded (best_set_aies_exchange): this rank moves `cnt` walkers of each half, partners come from the whole
        // other half, the moved slice is all-gathered after every half-step
        const int64_t cnt = st->aies_fn ? half / st->aies_world : half, off = st->aies_fn ? st->aies_rank * cnt : 0;
        tc::Run Rh = R;
        Rh.B = cnt;
        Rh.n_oth = half;
        for (int hh = 0; hh < 2; ++hh) {
          const int64_t half0 = hh == 0 ? 0 : half;
          Rh.own0 = half0 + off;
          Rh.oth0 = hh == 0 ? half : 0;
          BEST_TRY(launch_tc<tc::M_AIES>(ctx, Rh, cnt, s));
          if (st->aies_fn) BEST_TRY(aies_exchange(ctx, st, half0, s));
        }
      }
    }
    t0 += seg;
    if (adapt) BEST_TRY(adapt_window_rows(ctx, st, wb, seg, s));
  }
  if (method == tc::M_MH || method == tc::M_AIES) st->grad_valid = false;
  return BEST_OK;
}

}  // namespace best
