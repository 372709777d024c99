// Backward kernels (§8 a6-a7): persistent, warp-specialised, tcgen05 + TMEM, no atomics.
//
// The backward is split into two passes over the same (sequence, head, tile) work list so that
// every output tile is owned by exactly one CTA and accumulated in TMEM in a fixed order
// (deterministic by construction; DESIGN.md §5 discusses the 7-vs-5 GEMM trade):
//
//   kIsDQ = false  (dK/dV pass, KEY tile stationary):   X1 = K^, X2 = V ;  stream Y1 = Q^, Y2 = dO
//       S^T  = K^ Q^_sub^T      dP^T = V dO_sub^T         [128 keys x 64 queries] each
//       P^T  = exp2(S^T c - lse2[query])                   dS^T = P^T * (dP^T - delta[query])
//       dV  += P^T dO_sub       dK~ += dS^T Q^_sub         (A operand = P^T / dS^T in TMEM)
//   kIsDQ = true   (dQ pass, QUERY tile stationary):     X1 = Q^, X2 = dO ; stream Y1 = K^, Y2 = V
//       S    = Q^ K^_sub^T      dP   = dO V_sub^T         [128 queries x 64 keys] each
//       dS   = exp2(S - lse2[row]) * (dP - delta[row]) * sk
//       dQ~ += dS K^_sub
//
// The streamed 128-row tile is consumed in two 64-row halves so that S and dP can be double
// buffered in TMEM: acc0 [0,128) acc1 [128,256) S[2] at 256/320 dP[2] at 384/448 (= 512 columns).
// P / dS (bf16) alias the first half of the S / dP buffer they came from.
// No key masking is needed: prep zero-pads K^, V, Q^, dO tail rows and sets lse2 = +inf on padded
// query rows, so every padded element contributes exactly 0 to stored rows.
//
//   warp 4 producer (cp.async.bulk) | warp 5 MMA issuer | warps 0-3 one TMEM lane (row) per thread
#pragma once
#include "common.cuh"
#include "sm100.cuh"

namespace arachne {

struct BwdParams {
  const uint8_t* qt;       // Q^' fp16 images (q~ * softmax_scale * log2e)   [H][n_tiles][TILE]
  const uint8_t* kt;       // K^ fp16 images
  const uint8_t* vt;       // V  bf16 images
  const uint8_t* dot;      // dO bf16 images
  const float* lse2_t;     // [H][n_tiles][128]  lse*log2e, +inf on pad rows
  const float* delta_t;    // [H][n_tiles][128]
  float* gq_t;             // out: dl/dq~ fp32 [N,H,D]
  float* gk_t;             // out: dl/dk~ fp32 [N,H,D]
  ShardedPtr dv;           // out: bf16 [N,H_total,D], possibly sharded by token range (common.cuh)
};

template <int D>
struct BwdCfg {
  static constexpr int kTileBytes = kTileRows * D * 2;
  static constexpr int kStages = (D == 128) ? 2 : 4;
  static constexpr int kNumBars = 2 + 2 * kStages + 2 + 2 + 2;
  static constexpr int kSmemBytes = kTileBytes * (2 + 2 * kStages) + kStages * 1024 + 8 * kNumBars + 16 + 1024;
  static constexpr uint32_t kColAcc0 = 0, kColAcc1 = 128, kColS = 256, kColDP = 384;
};

template <int D, bool kIsDQ>
__global__ void __launch_bounds__(192, 1) bwd_kernel(ProblemDesc pd, BwdParams bp, int counter_slot) {
  using Cfg = BwdCfg<D>;
  constexpr int TILE = Cfg::kTileBytes;
  constexpr int STAGES = Cfg::kStages;
  constexpr uint32_t BLK = kTileRows * 128;   // bytes of one 64-element block of a tile image
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sX1 = smem;
  uint8_t* sX2 = sX1 + TILE;
  uint8_t* sY1 = sX2 + TILE;
  uint8_t* sY2 = sY1 + STAGES * TILE;
  float* sLse = reinterpret_cast<float*>(sY2 + STAGES * TILE);    // [STAGES][128]
  float* sDelta = sLse + STAGES * 128;                             // [STAGES][128]
  uint64_t* bars = reinterpret_cast<uint64_t*>(sDelta + STAGES * 128);
  uint64_t* x_full = bars;
  uint64_t* x_empty = bars + 1;
  uint64_t* y_full = bars + 2;            // [STAGES]
  uint64_t* y_empty = y_full + STAGES;    // [STAGES]
  uint64_t* sdp_full = y_empty + STAGES;  // [2] MMA -> compute
  uint64_t* pds_full = sdp_full + 2;      // [2] compute (128) -> MMA
  uint64_t* acc_done = pds_full + 2;      // MMA -> compute (epilogue)
  uint64_t* acc_free = acc_done + 1;      // compute (128) -> MMA
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_free + 1);
  (void)counter_slot;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(x_full, 1); mbar_init(x_empty, 1);
    for (int s = 0; s < STAGES; ++s) { mbar_init(&y_full[s], 1); mbar_init(&y_empty[s], 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(&sdp_full[s], 1); mbar_init(&pds_full[s], 128); }
    mbar_init(acc_done, 1);
    mbar_init(acc_free, 128);
    fence_mbar_init();
  }
  if (warp == 5) { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const size_t head_stride = static_cast<size_t>(pd.n_tiles_total) * TILE;
  const uint8_t* gX1 = kIsDQ ? bp.qt : bp.kt;
  const uint8_t* gX2 = kIsDQ ? bp.dot : bp.vt;
  const uint8_t* gY1 = kIsDQ ? bp.kt : bp.qt;
  const uint8_t* gY2 = kIsDQ ? bp.vt : bp.dot;

  if (warp == 4) {
    // ------------------------------------------------------------------ producer
    if (lane == 0) {
      uint32_t it = 0, yt = 0;
      for (int item = pd.item_ptr[blockIdx.x]; item < pd.item_ptr[blockIdx.x + 1]; ++item, ++it) {
        const WorkItem wi = pd.items[item];
        const SeqInfo sq = pd.seqs[wi.seq];
        const size_t hoff = wi.head * head_stride;
        const size_t xoff = hoff + static_cast<size_t>(sq.tile_base + wi.tile) * TILE;
        mbar_wait(x_empty, (it & 1) ^ 1);
        mbar_expect_tx(x_full, 2 * TILE);
        bulk_g2s(sX1, gX1 + xoff, TILE, x_full);
        bulk_g2s(sX2, gX2 + xoff, TILE, x_full);
        for (int j = 0; j < sq.n_tiles; ++j, ++yt) {
          const uint32_t st = yt % STAGES, ph = (yt / STAGES) & 1;
          const size_t yoff = hoff + static_cast<size_t>(sq.tile_base + j) * TILE;
          mbar_wait(&y_empty[st], ph ^ 1);
          mbar_expect_tx(&y_full[st], 2 * TILE + (kIsDQ ? 0 : 1024));
          bulk_g2s(sY1 + st * TILE, gY1 + yoff, TILE, &y_full[st]);
          bulk_g2s(sY2 + st * TILE, gY2 + yoff, TILE, &y_full[st]);
          if (!kIsDQ) {
            const size_t roff = (static_cast<size_t>(wi.head) * pd.n_tiles_total + sq.tile_base + j) * kTileRows;
            bulk_g2s(sLse + st * 128, bp.lse2_t + roff, 512, &y_full[st]);
            bulk_g2s(sDelta + st * 128, bp.delta_t + roff, 512, &y_full[st]);
          }
        }
      }
    }
  } else if (warp == 5) {
    // ------------------------------------------------------------------ MMA issuer (whole warp convergent,
    // one elected lane issues: keeps descriptors in uniform registers, no per-instruction election loop)
    {
      // S from the forward's fp16 Q^', K^ images; dS fp16 (scaled by the group's sk); P, V, dO bf16
      constexpr uint32_t idesc_s = make_idesc(128, 64, FMT_F16, FMT_F16, MAJOR_K, MAJOR_K);
      constexpr uint32_t idesc_dp = make_idesc(128, 64, FMT_BF16, FMT_BF16, MAJOR_K, MAJOR_K);
      constexpr uint32_t idesc_pv = make_idesc(128, D, FMT_BF16, FMT_BF16, MAJOR_K, MAJOR_MN);
      constexpr uint32_t idesc_ds = make_idesc(128, D, FMT_F16, FMT_F16, MAJOR_K, MAJOR_MN);
      const uint32_t aX1 = smem_u32(sX1), aX2 = smem_u32(sX2), aY1 = smem_u32(sY1), aY2 = smem_u32(sY2);
      const uint32_t tAcc0 = tbase + Cfg::kColAcc0, tAcc1 = tbase + Cfg::kColAcc1;
      uint32_t it = 0, yt = 0, g = 0;
      // S/dP of sub-iteration gg: streamed tile `ytile` (global counter), half u
      auto issue_sdp = [&](uint32_t gg, uint32_t ytile, uint32_t u) {
        const uint32_t st = ytile % STAGES, ph = (ytile / STAGES) & 1;
        if (u == 0) { mbar_wait(&y_full[st], ph); tc_fence_after(); }
        const uint32_t tS = tbase + Cfg::kColS + (gg & 1) * 64, tdP = tbase + Cfg::kColDP + (gg & 1) * 64;
        const uint32_t yb = st * TILE + u * 8192;      // rows 64u.. of the streamed image
        if (elect_one()) {
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t koff = (kk >> 2) * BLK + (kk & 3) * 32;
          umma_ss(tS, make_sdesc(aX1 + koff, 16, 1024), make_sdesc(aY1 + yb + koff, 16, 1024), idesc_s, kk > 0);
        }
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t koff = (kk >> 2) * BLK + (kk & 3) * 32;
          umma_ss(tdP, make_sdesc(aX2 + koff, 16, 1024), make_sdesc(aY2 + yb + koff, 16, 1024), idesc_dp, kk > 0);
        }
        umma_commit(&sdp_full[gg & 1]);
        }
        __syncwarp();
      };
      for (int item = pd.item_ptr[blockIdx.x]; item < pd.item_ptr[blockIdx.x + 1]; ++item, ++it) {
        const WorkItem wi = pd.items[item];
        const uint32_t G = 2u * pd.seqs[wi.seq].n_tiles;
        mbar_wait(x_full, it & 1);
        tc_fence_after();
        issue_sdp(g, yt, 0);
        for (uint32_t s = 0; s < G; ++s) {
          const uint32_t gg = g + s, u = s & 1, ytile = yt + (s >> 1), st = ytile % STAGES;
          if (s + 1 < G) issue_sdp(gg + 1, yt + ((s + 1) >> 1), (s + 1) & 1);
          else { if (elect_one()) umma_commit(x_empty); __syncwarp(); }
          if (s == 0) mbar_wait(acc_free, (it & 1) ^ 1);
          mbar_wait(&pds_full[gg & 1], (gg >> 1) & 1);
          tc_fence_after();
          const uint32_t tP = tbase + Cfg::kColS + (gg & 1) * 64, tdS = tbase + Cfg::kColDP + (gg & 1) * 64;
          if (elect_one()) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            const uint32_t roff = st * TILE + (u * 64 + kk * 16) * 128;     // K rows of the MN-major B operand
            const uint32_t acc = (s > 0 || kk > 0) ? 1u : 0u;
            if (!kIsDQ) {
              umma_ts(tAcc0, tP + kk * 8, make_sdesc(aY2 + roff, BLK, 1024), idesc_pv, acc);    // dV += P^T dO
              umma_ts(tAcc1, tdS + kk * 8, make_sdesc(aY1 + roff, BLK, 1024), idesc_ds, acc);   // dK~ += dS^T Q^'
            } else {
              umma_ts(tAcc0, tdS + kk * 8, make_sdesc(aY1 + roff, BLK, 1024), idesc_ds, acc);   // dQ~ += dS K^
            }
          }
          if (u == 1) umma_commit(&y_empty[st]);
          }
          __syncwarp();
        }
        if (elect_one()) umma_commit(acc_done);
        __syncwarp();
        g += G;
        yt += G >> 1;
      }
    }
  } else {
    // ------------------------------------------------------------------ compute + epilogue (warps 0-3)
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
    const int row = threadIdx.x;
    uint32_t it = 0, yt = 0, g = 0;
    for (int item = pd.item_ptr[blockIdx.x]; item < pd.item_ptr[blockIdx.x + 1]; ++item, ++it) {
      const WorkItem wi = pd.items[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      const uint32_t G = 2u * sq.n_tiles;
      const float2 skv = *reinterpret_cast<const float2*>(pd.grp_sk + (static_cast<size_t>(wi.seq) * pd.H + wi.head) * 2);
      const float sk = skv.x;                    // dS is rounded to fp16 as dS * sk (delta already carries sk: bwd_scale_kernel)
      float lse2_r = 0.f, delta_r = 0.f;
      if (kIsDQ) {
        const size_t roff = (static_cast<size_t>(wi.head) * pd.n_tiles_total + sq.tile_base + wi.tile) * kTileRows + row;
        lse2_r = bp.lse2_t[roff];
        delta_r = bp.delta_t[roff];
      }
      for (uint32_t s = 0; s < G; ++s) {
        const uint32_t gg = g + s, u = s & 1, ytile = yt + (s >> 1), st = ytile % STAGES;
        if (!kIsDQ && u == 0) mbar_wait(&y_full[st], (ytile / STAGES) & 1);   // lse2/delta of the streamed rows
        mbar_wait(&sdp_full[gg & 1], (gg >> 1) & 1);
        tc_fence_after();
        const uint32_t tS = tbase + Cfg::kColS + (gg & 1) * 64 + lane_base;
        const uint32_t tdP = tbase + Cfg::kColDP + (gg & 1) * 64 + lane_base;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t sv[32], dpv[32];
          tmem_ld32(tS + half * 32, sv);
          tmem_ld32(tdP + half * 32, dpv);
          tmem_wait_ld();
          uint32_t pp[16], dd[16];
#pragma unroll
          for (int c = 0; c < 32; c += 2) {
            float l0, l1, d0, d1;
            if (kIsDQ) { l0 = l1 = lse2_r; d0 = d1 = delta_r; }
            else {
              const int col = u * 64 + half * 32 + c;
              const float2 lv = *reinterpret_cast<const float2*>(&sLse[st * 128 + col]);
              const float2 dv2 = *reinterpret_cast<const float2*>(&sDelta[st * 128 + col]);
              l0 = lv.x; l1 = lv.y; d0 = dv2.x; d1 = dv2.y;
            }
            const float p0 = ex2_approx(__uint_as_float(sv[c]) - l0);        // S is already in the exp2 domain (Q^')
            const float p1 = ex2_approx(__uint_as_float(sv[c + 1]) - l1);
            const float ds0 = p0 * fmaf(__uint_as_float(dpv[c]), sk, -d0);
            const float ds1 = p1 * fmaf(__uint_as_float(dpv[c + 1]), sk, -d1);
            pp[c >> 1] = pack_bf16x2(p0, p1);
            dd[c >> 1] = pack_f16x2(ds0, ds1);
          }
          if (!kIsDQ) tmem_st16(tS + half * 16, pp);
          tmem_st16(tdP + half * 16, dd);
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(&pds_full[gg & 1]);
      }
      // ---- epilogue
      mbar_wait(acc_done, it & 1);
      tc_fence_after();
      const int n = wi.tile * kTileRows + row;
      const bool valid_row = n < sq.len;
      const size_t out_off = (static_cast<size_t>(sq.tok_start + n) * pd.H + wi.head) * D;
      const uint32_t tA0 = tbase + Cfg::kColAcc0 + lane_base, tA1 = tbase + Cfg::kColAcc1 + lane_base;
      // dq~ = scale * dS k~;  dk~ = scale * dS^T q~ = ln2 * dS^T Q^';  dS carries sk
      const float sc = (kIsDQ ? pd.softmax_scale : 0.6931471805599453f) * skv.y;
      __nv_bfloat16* dv_row = valid_row ? raw_row<__nv_bfloat16>(pd.sh, bp.dv, sq.tok_start + n, wi.head, D) : nullptr;
      float* gout = (kIsDQ ? bp.gq_t : bp.gk_t) + out_off;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t a[32];
        tmem_ld32((kIsDQ ? tA0 : tA1) + c * 32, a);
        tmem_wait_ld();
        if (valid_row) {
#pragma unroll
          for (int i = 0; i < 32; i += 4) {
            float4 f;
            f.x = __uint_as_float(a[i]) * sc; f.y = __uint_as_float(a[i + 1]) * sc;
            f.z = __uint_as_float(a[i + 2]) * sc; f.w = __uint_as_float(a[i + 3]) * sc;
            *reinterpret_cast<float4*>(gout + c * 32 + i) = f;
          }
        }
        if (!kIsDQ) {
          tmem_ld32(tA0 + c * 32, a);
          tmem_wait_ld();
          if (valid_row) {
#pragma unroll
            for (int i = 0; i < 32; i += 8) {
              uint4 w;
              w.x = pack_bf16x2(__uint_as_float(a[i]), __uint_as_float(a[i + 1]));
              w.y = pack_bf16x2(__uint_as_float(a[i + 2]), __uint_as_float(a[i + 3]));
              w.z = pack_bf16x2(__uint_as_float(a[i + 4]), __uint_as_float(a[i + 5]));
              w.w = pack_bf16x2(__uint_as_float(a[i + 6]), __uint_as_float(a[i + 7]));
              *reinterpret_cast<uint4*>(dv_row + c * 32 + i) = w;
            }
          }
        }
      }
      tc_fence_before();
      mbar_arrive(acc_free);
      g += G;
      yt += G >> 1;
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 5) tmem_dealloc(tbase, 512);
}

}  // namespace arachne
