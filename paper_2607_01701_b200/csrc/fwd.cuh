// Forward kernel (§8 a2-a4): persistent, warp-specialised, tcgen05 + TMEM.
//
// Work item = (sequence b, head h, 128-row query tile).  Per item the CTA streams the
// ceil(L_b/128) key/value tiles of sequence b ONLY (block-diagonal: no other tile is ever
// touched, no masked-out tile is computed):
//
//   warp 4 (1 lane)  producer : cp.async.bulk  Q^ image, then K^_j / V_j images into a ring
//   warp 5 (1 lane)  MMA      : S_j = Q^ K^_j^T   (SS, fp16 x fp16 -> fp32 TMEM, double-buffered)
//                               O  += P_j V_j     (TS: P_j bf16 in TMEM aliasing S_j; V MN-major)
//   warps 0-3        softmax  : one query row per thread: tcgen05.ld S row, online softmax in the
//                               exp2 domain with LAZY rescaling (O is only rescaled when the row
//                               max grew by > 2^8; QK-RMSNorm bounds the logits so this is rare),
//                               P -> bf16 -> tcgen05.st, final O / l -> bf16, LSE -> fp32.
//
// Q^, K^ are fp16 (RMSNorm bounds |x^_d| <= gamma_max * sqrt(D)); fp16 operands put the LSE
// error floor at ~2e-4 instead of ~1.5e-3 for bf16.  P and V are bf16.
#pragma once
#include "common.cuh"
#include "sm100.cuh"

namespace arachne {

struct FwdParams {
  const uint8_t* qt;      // [H][n_tiles][TILE_BYTES]  Q^ fp16 images
  const uint8_t* kt;      // K^ fp16 images
  const uint8_t* vt;      // V bf16 images
  __nv_bfloat16* o;       // [N,H,D]
  float* lse;             // [H,N]
};

template <int D>
struct FwdCfg {
  static constexpr int kTileBytes = kTileRows * D * 2;
  static constexpr int kStages = (D == 128) ? 3 : 4;
  static constexpr int kNumBars = 2 + 4 * kStages + 2 + 2 + 2;
  static constexpr int kSmemBytes = kTileBytes * (1 + 2 * kStages) + 8 * kNumBars + 16 + 1024;
  static constexpr int kThreads = 192;
  // TMEM columns: S0 [0,128) S1 [128,256) O [256, 256+D)
  static constexpr uint32_t kColS0 = 0, kColS1 = 128, kColO = 256;
};

template <int D>
__global__ void __launch_bounds__(192, 1) fwd_kernel(ProblemDesc pd, FwdParams fp) {
  using Cfg = FwdCfg<D>;
  constexpr int TILE = Cfg::kTileBytes;
  constexpr int STAGES = Cfg::kStages;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* sQ = smem;
  uint8_t* sK = sQ + TILE;
  uint8_t* sV = sK + STAGES * TILE;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sV + STAGES * TILE);
  uint64_t* q_full = bars;            // producer -> MMA
  uint64_t* q_empty = bars + 1;       // MMA (commit) -> producer
  uint64_t* k_full = bars + 2;        // [STAGES]
  uint64_t* k_empty = k_full + STAGES;
  uint64_t* v_full = k_empty + STAGES;
  uint64_t* v_empty = v_full + STAGES;
  uint64_t* s_full = v_empty + STAGES;   // [2] MMA (commit) -> softmax
  uint64_t* p_full = s_full + 2;         // [2] softmax (128 arrivals) -> MMA
  uint64_t* pv_done = p_full + 2;        // MMA (commit) -> softmax: one phase per PV
  uint64_t* o_free = pv_done + 1;        // softmax epilogue (128 arrivals) -> MMA
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(o_free + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    mbar_init(q_full, 1); mbar_init(q_empty, 1);
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(&k_full[s], 1); mbar_init(&k_empty[s], 1);
      mbar_init(&v_full[s], 1); mbar_init(&v_empty[s], 1);
    }
    for (int s = 0; s < 2; ++s) { mbar_init(&s_full[s], 1); mbar_init(&p_full[s], 128); }
    mbar_init(pv_done, 1);
    mbar_init(o_free, 128);
    fence_mbar_init();
  }
  if (warp == 5) { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const float scale_log2 = pd.softmax_scale * 1.4426950408889634f;
  const size_t head_stride = static_cast<size_t>(pd.n_tiles_total) * TILE;

  if (warp == 4) {
    // ------------------------------------------------------------------ producer
    if (lane == 0) {
      uint32_t it = 0, kv = 0;
      for (int item = blockIdx.x; item < pd.n_items; item += gridDim.x, ++it) {
        const WorkItem wi = pd.items[item];
        const SeqInfo sq = pd.seqs[wi.seq];
        const uint8_t* hbase_q = fp.qt + wi.head * head_stride;
        const uint8_t* hbase_k = fp.kt + wi.head * head_stride;
        const uint8_t* hbase_v = fp.vt + wi.head * head_stride;
        mbar_wait(q_empty, (it & 1) ^ 1);
        mbar_expect_tx(q_full, TILE);
        bulk_g2s(sQ, hbase_q + static_cast<size_t>(sq.tile_base + wi.tile) * TILE, TILE, q_full);
        for (int j = 0; j < sq.n_tiles; ++j, ++kv) {
          const uint32_t st = kv % STAGES, ph = (kv / STAGES) & 1;
          const size_t off = static_cast<size_t>(sq.tile_base + j) * TILE;
          mbar_wait(&k_empty[st], ph ^ 1);
          mbar_expect_tx(&k_full[st], TILE);
          bulk_g2s(sK + st * TILE, hbase_k + off, TILE, &k_full[st]);
          mbar_wait(&v_empty[st], ph ^ 1);
          mbar_expect_tx(&v_full[st], TILE);
          bulk_g2s(sV + st * TILE, hbase_v + off, TILE, &v_full[st]);
        }
      }
    }
  } else if (warp == 5) {
    // ------------------------------------------------------------------ MMA issuer
    // The whole warp runs the loop convergently (uniform descriptors -> plain UTCHMMA issue, no
    // per-instruction election loop); one elected lane issues the tcgen05 instructions.
    {
      constexpr uint32_t idesc_s = make_idesc(128, 128, FMT_F16, FMT_F16, MAJOR_K, MAJOR_K);
      constexpr uint32_t idesc_o = make_idesc(128, D, FMT_BF16, FMT_BF16, MAJOR_K, MAJOR_MN);
      const uint32_t aQ = smem_u32(sQ), aK = smem_u32(sK), aV = smem_u32(sV);
      const uint32_t tS[2] = {tbase + Cfg::kColS0, tbase + Cfg::kColS1};
      const uint32_t tO = tbase + Cfg::kColO;
      uint32_t it = 0, kv = 0;   // kv: global count of S tiles issued == global tile counter
      auto issue_s = [&](uint32_t g) {
        const uint32_t st = g % STAGES, ph = (g / STAGES) & 1;
        mbar_wait(&k_full[st], ph);
        tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint32_t koff = (kk >> 2) * (kTileRows * 128) + (kk & 3) * 32;
            umma_ss(tS[g & 1], make_sdesc(aQ + koff, 16, 1024), make_sdesc(aK + st * TILE + koff, 16, 1024),
                    idesc_s, kk > 0);
          }
          umma_commit(&k_empty[st]);
          umma_commit(&s_full[g & 1]);
        }
        __syncwarp();
      };
      for (int item = blockIdx.x; item < pd.n_items; item += gridDim.x, ++it) {
        const WorkItem wi = pd.items[item];
        const int n_kv = pd.seqs[wi.seq].n_tiles;
        mbar_wait(q_full, it & 1);
        issue_s(kv);
        for (int j = 0; j < n_kv; ++j) {
          const uint32_t g = kv + j;
          if (j + 1 < n_kv) issue_s(g + 1);
          else { if (elect_one()) umma_commit(q_empty); __syncwarp(); }   // all S MMAs of this item issued: Q^ smem reusable once they finish
          const uint32_t st = g % STAGES, ph = (g / STAGES) & 1;
          mbar_wait(&v_full[st], ph);
          if (j == 0) mbar_wait(o_free, (it & 1) ^ 1);     // previous item's epilogue has drained O
          mbar_wait(&p_full[g & 1], (g >> 1) & 1);
          tc_fence_after();
          if (elect_one()) {
#pragma unroll
            for (int kk = 0; kk < kTileRows / 16; ++kk) {
              umma_ts(tO, tS[g & 1] + kk * 8, make_sdesc(aV + st * TILE + kk * 2048, kTileRows * 128, 1024),
                      idesc_o, (j > 0 || kk > 0) ? 1u : 0u);
            }
            umma_commit(&v_empty[st]);
            umma_commit(pv_done);
          }
          __syncwarp();
        }
        kv += n_kv;
      }
    }
  } else {
    // ------------------------------------------------------------------ softmax + epilogue (warps 0-3)
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;   // this warp's TMEM lanes
    const uint32_t tS[2] = {tbase + Cfg::kColS0 + lane_base, tbase + Cfg::kColS1 + lane_base};
    const uint32_t tO = tbase + Cfg::kColO + lane_base;
    const int row = threadIdx.x;   // query row inside the tile
    uint32_t g = 0;                // global S/PV tile counter (matches the MMA warp's)
    for (int item = blockIdx.x; item < pd.n_items; item += gridDim.x) {
      const WorkItem wi = pd.items[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      float m = -INFINITY, l = 0.f;
      for (int j = 0; j < sq.n_tiles; ++j, ++g) {
        mbar_wait(&s_full[g & 1], (g >> 1) & 1);
        tc_fence_after();
        uint32_t su[128];
#pragma unroll
        for (int c = 0; c < 4; ++c) tmem_ld32(tS[g & 1] + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&su[c * 32]));
        tmem_wait_ld();
        const int valid = sq.len - j * kTileRows;    // keys of this tile that exist
        if (valid < kTileRows) {
#pragma unroll
          for (int c = 0; c < 128; ++c) if (c >= valid) su[c] = 0xff800000u;   // -inf
        }
        float mx = __uint_as_float(su[0]);
#pragma unroll
        for (int c = 1; c < 128; ++c) mx = fmaxf(mx, __uint_as_float(su[c]));
        const float m_new = fmaxf(m, mx * scale_log2);
        float alpha = 1.0f;
        // lazy rescale: keep the stale max unless it is more than 8 (log2 units) too small
        const bool bump = (m_new - m) > 8.0f;     // true on the first tile (m = -inf)
        if (bump) { alpha = ex2_approx(m - m_new); m = m_new; }
        float rs = 0.f;
        uint32_t pk[64];
#pragma unroll
        for (int c = 0; c < 128; c += 2) {
          const float p0 = ex2_approx(fmaf(__uint_as_float(su[c]), scale_log2, -m));
          const float p1 = ex2_approx(fmaf(__uint_as_float(su[c + 1]), scale_log2, -m));
          rs += p0 + p1;
          pk[c >> 1] = pack_bf16x2(p0, p1);
        }
        l = l * alpha + rs;
        tmem_st32(tS[g & 1], *reinterpret_cast<uint32_t(*)[32]>(&pk[0]));
        tmem_st32(tS[g & 1] + 32, *reinterpret_cast<uint32_t(*)[32]>(&pk[32]));
        if (j > 0 && __any_sync(0xffffffffu, bump)) {
          // O += P V of tile g-1 must have completed before O is rescaled
          mbar_wait(pv_done, (g - 1) & 1);
          tc_fence_after();
#pragma unroll
          for (int c = 0; c < D / 32; ++c) {
            uint32_t o[32];
            tmem_ld32(tO + c * 32, o);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
            tmem_st32(tO + c * 32, o);
          }
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(&p_full[g & 1]);
      }
      // ---- epilogue: O / l -> bf16, LSE (natural log, reading R9)
      mbar_wait(pv_done, (g - 1) & 1);
      tc_fence_after();
      const int n = wi.tile * kTileRows + row;     // token inside the sequence
      const bool valid_row = n < sq.len;
      const float inv_l = 1.0f / l;
      __nv_bfloat16* orow = fp.o + (static_cast<size_t>(sq.tok_start + n) * pd.H + wi.head) * D;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        tmem_ld32(tO + c * 32, o);
        tmem_wait_ld();
        if (valid_row) {
#pragma unroll
          for (int i = 0; i < 32; i += 8) {
            uint4 u;
            u.x = pack_bf16x2(__uint_as_float(o[i]) * inv_l, __uint_as_float(o[i + 1]) * inv_l);
            u.y = pack_bf16x2(__uint_as_float(o[i + 2]) * inv_l, __uint_as_float(o[i + 3]) * inv_l);
            u.z = pack_bf16x2(__uint_as_float(o[i + 4]) * inv_l, __uint_as_float(o[i + 5]) * inv_l);
            u.w = pack_bf16x2(__uint_as_float(o[i + 6]) * inv_l, __uint_as_float(o[i + 7]) * inv_l);
            *reinterpret_cast<uint4*>(orow + c * 32 + i) = u;
          }
        }
      }
      if (valid_row)
        fp.lse[static_cast<size_t>(wi.head) * pd.N + sq.tok_start + n] = (m + log2f(l)) * 0.6931471805599453f;
      tc_fence_before();
      mbar_arrive(o_free);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 5) tmem_dealloc(tbase, 512);
}

}  // namespace arachne
