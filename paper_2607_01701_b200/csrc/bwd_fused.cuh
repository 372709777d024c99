// Fused single-pass backward (§8 a6 + a7): 5 GEMMs per (key tile, query tile) pair, dK/dV accumulated in TMEM across
// the query loop, dQ~ partial tiles reduced into a blocked fp32 accumulator in global memory by the TMA engine
// (cp.reduce.async.bulk .add at L2).  Default: fp32 additions in arrival order -> run-to-run bit differences;
// ARACHNE_FLAG_DETERMINISTIC: the same kernel, the partial tiles reduced as FIXED-POINT int32 ("order-independent reduction"
// below): integer addition is associative, so the result no longer depends on the order at all.
//
// Work item = (sequence b, head h, 128-row KEY tile).
// Items are taken DYNAMICALLY from the plan's LPT-ordered list: lane 0 of the producer warp does an atomicAdd on a per-launch
// counter and hands the index to the other warp roles through a 4-slot shared-memory ring (sm100.cuh, ItemRing).  The CTA keeps K^ and V of the tile in shared
// memory and streams the ceil(L_b/128) QUERY tiles of sequence b only (block-diagonal):
//
//   S^T  = K^  Q^_i^T        SS   [128 keys x 128 queries] fp32 -> TMEM cols [0,128)
//   dP^T = V   dO_i^T        SS                                  -> TMEM cols [128,256)
//   P^T  = exp2(S^T - lse2[query])              bf16, written back over S^T (A operand of dV)
//   dS^T = P^T * (dP^T - delta[query]) * sk     fp16, written to shared memory (one tile image); sk: prep.cuh
//   dV  += P^T  dO_i         TS   acc TMEM cols [256,256+D)
//   dK~ += dS^T Q^_i         SS   acc TMEM cols [256+D,256+2D)   (A = dS^T image, K-major)
//   dQ~_i = dS  K^           SS   -> TMEM cols [128,256) (aliases dP^T) (A = dS^T image, MN-major)
//
// TMEM is full (512 columns), so dQ~_i shares its columns with dP^T; the MMA issue order
//   S_0 P_0 V_0 S_1 | Q_0 K_0 P_1 V_1 S_2 | Q_1 K_1 P_2 V_2 S_3 | ...
// gives the drain of dQ~_i one GEMM (K_i) of slack before P_{i+1} needs the columns, lets the exp
// of tile i+1 overlap Q_i/K_i, and needs only ONE dO stage and TWO Q^ stages in shared memory.
//
// Warps: 0-3 and 4-7 compute (warp w owns TMEM lanes 32*(w%4)..; warps 0-3 take query columns
// [0,64), warps 4-7 [64,128)); 8-11 drain dQ~ (TMEM -> registers -> staging smem -> bulk
// reduce-add); 12 producer (cp.async.bulk); 13 MMA issuer (whole warp convergent, elected lane issues).
#pragma once
#include "common.cuh"
#include "rawtile.cuh"
#include "sm100.cuh"

namespace arachne {

struct BwdFusedParams {
  const uint8_t* qt;       // Q^' fp16 images (q~ * softmax_scale * log2e)   [H][n_tiles][TILE]
  const uint8_t* kt;       // K^ fp16 images
  const uint8_t* vt;       // V  bf16 images   (only when v_raw.base == nullptr)
  const uint8_t* dot;      // dO bf16 images   (only when do_raw.base == nullptr)
  RawTensor v_raw, do_raw; // base != nullptr: V / dO tiles come straight from the raw tensors by tensor-map TMA (rawtile.cuh)
  const float* lse2_t;     // [H][n_tiles][128]  lse*log2e, +inf on pad rows
  const float* delta_t;    // [H][n_tiles][128]
  float* gq_blk;           // in/out: dl/dq~ fp32, blocked [H][n_tiles][D/32][128][32], 16-byte pieces
                           //         XOR-swizzled with (row & 7); zeroed by prep_kernel
  float* gk_t;             // out: dl/dk~ fp32 [N,H,D]
  ShardedPtr dv;           // out: bf16 [N,H_total,D], possibly sharded by token range (common.cuh)
  float* gv_t;             // nullable (context parallelism): dV PARTIAL fp32 [N,H,D] written instead of dv
  int dq_fixed;            // ARACHNE_FLAG_DETERMINISTIC: gq_blk is an int32 fixed-point accumulator (see below)
  float* rowqs_t;          // dq_fixed: [H][n_tiles][128] fixed-point scale of every query row (bwd_scale_kernel); a drain thread
                           // overwrites its row's entry with NaN when a partial is non-finite or out of range
};

// Order-independent (deterministic) dq~ reduction.  The L2 reduce-add of fp32 partial tiles is associative only up to rounding,
// so the default mode is not bit-reproducible.  With ARACHNE_FLAG_DETERMINISTIC every partial value is converted to FIXED POINT
// — round-to-nearest of value * qs_i, qs_i a power of two per QUERY ROW i (per (token, head)) — and reduced with the INTEGER
// form of the same bulk operation (cp.reduce.async.bulk .add.s32): integer addition is exactly associative and commutative, so
// the sum is the same whatever order the 148 CTAs' reductions reach L2 in; post_kernel multiplies by 1 / qs_i.  Same bytes,
// same schedule and the same speed as the default mode, and no reliance on cross-SM ordering of asynchronous reductions (an
// earlier ticket scheme that serialised the fp32 additions by key tile was 5 % slower and, one run in ten at head_dim 64, let
// one reduction overtake another: profiles/r2_deterministic.md).
//   qs_i comes from a rigorous bound, so no partial sum can overflow in ANY order: with P_ij >= 0, sum_j P_ij = 1,
//     sum_j |dS_ij| = sum_j P_ij |dO_i.V_j - dO_i.O_i| <= 2 |dO_i| max_j|V_j|                 (O_i is a convex combination of the V_j)
//     sum over all keys of |dS_ij k~_j[d]| <= 2 |dO_i| max|V| max_j|k~_j| =: B_i,   |k~_j|^2 <= D max_d gamma_k[d]^2 under RMSNorm
//   (|dO_i| and the group's max|V| come from prep_kernel), and qs_i = 2^floor(log2(2^30 / (1.01 softmax_scale B_i))) (bwd_scale_kernel).
//   The price is precision, not range: the quantum of row i is B_i * 2^-30, i.e. ~2^-13 .. 2^-17 of a typical element of THAT
//   row whatever its size (measured dQ rel-L2 against the oracle: same 1.7e-3 as the fp32 mode, profiles/r2_deterministic.md).
//   Because the scale follows the row's own |dO_i|, a token with an outlying upstream gradient costs the other rows nothing
//   (a scale per (sequence, head) group, as in round 2, left them log2(outlier / typical) bits short).  What still costs bits
//   is an outlying VALUE row: max_j|V_j| enters every row's bound, because any row may attend to it; a V row 2^k above typical
//   takes k of the ~13-17 spare bits from every row of its (sequence, head) group (tests/test_gpu_parity.py, heavy-tailed case).
//   The bound needs sum_j P_ij = 1, i.e. the LSE passed to the backward must be the forward's for the same inputs (the ABI's
//   precondition).  A partial that is non-finite or beyond 2^30 after scaling — NaN / inf in the inputs, or an LSE so foreign
//   that a single tile already breaks the bound — is not silently wrapped or dropped (cvt.rni.s32 turns NaN into 0): the drain
//   thread overwrites the row's scale with NaN and post_kernel emits NaN for that dQ row, as the fp32 mode would.  A foreign
//   LSE whose tiles each stay in range but whose SUM leaves int32 cannot be seen by anybody (the additions happen in L2).

template <int D>
struct BwdFusedCfg {
  static constexpr int kTileBytes = kTileRows * D * 2;
  static constexpr int kQStages = (D == 128) ? 2 : 4;
  static constexpr int kDOStages = (D == 128) ? 1 : 2;
  static constexpr int kDSBytes = kTileRows * kTileRows * 2;      // dS^T image, 128 x 128 bf16
  static constexpr int kStageBytes = kTileRows * 64 * 4;           // dQ~ staging: 128 rows x 64 fp32
  static constexpr int kNumBars = 2 + 2 * kQStages + 2 * kDOStages + 9 + 2 * kItemRing;
  static constexpr int kSmemBytes = kTileBytes * (2 + kQStages + kDOStages) + kDSBytes + kStageBytes +
                                    kQStages * 1024 + 8 * kNumBars + 16 + 4 * kItemRing;
  static constexpr int kThreads = 512;   // 4 warpgroups: compute, compute, dQ~ drain, {producer, MMA, 2 idle warps}
  static constexpr uint32_t kColS = 0, kColDP = 128, kColDV = 256, kColDK = 256 + D;
};

// offset (in floats) of element (row q, column d) inside one blocked dq~ tile
__host__ __device__ __forceinline__ uint32_t gq_blk_off(int q, int d) {
  return static_cast<uint32_t>(d >> 5) * (kTileRows * 32) + q * 32 + ((((d & 31) >> 2) ^ (q & 7)) << 2) + (d & 3);
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}
// Register re-allocation between warpgroups (512 threads x 128 = the whole register file): the producer / MMA
// warpgroup gives registers back and the drain warpgroup takes them (no spills anywhere in the kernel).  Holding a
// whole 128 x D fp32 dQ~ tile in registers to release the TMEM columns before staging was tried and is slower
// (profiles/r1_notes.md §8): the dQ~ columns are not what the tensor pipe waits for.
template <int N>
__device__ __forceinline__ void setmaxnreg_inc() {
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void bulk_wait_group() {
  asm volatile("cp.async.bulk.wait_group %0;\n" ::"n"(N) : "memory");
}

template <int D>
__global__ void __launch_bounds__(512, 1) bwd_fused_kernel(ProblemDesc pd, BwdFusedParams bp, const __grid_constant__ RawMaps vmaps,
                                                            const __grid_constant__ RawMaps domaps) {
  using Cfg = BwdFusedCfg<D>;
  constexpr int TILE = Cfg::kTileBytes;
  constexpr int QS = Cfg::kQStages, DS = Cfg::kDOStages;
  constexpr uint32_t BLK = kTileRows * 128;   // bytes of one 64-element block of a tile image
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* sK = smem;
  uint8_t* sV = sK + TILE;
  uint8_t* sQ = sV + TILE;
  uint8_t* sdO = sQ + QS * TILE;
  uint8_t* sdS = sdO + DS * TILE;
  uint8_t* sStage = sdS + Cfg::kDSBytes;
  float* sLse = reinterpret_cast<float*>(sStage + Cfg::kStageBytes);   // [QS][128]
  float* sDelta = sLse + QS * 128;                                      // [QS][128]
  uint64_t* bars = reinterpret_cast<uint64_t*>(sDelta + QS * 128);
  uint64_t* kv_full = bars;                // producer -> MMA
  uint64_t* kv_free = bars + 1;            // MMA (commit) -> producer
  uint64_t* q_full = bars + 2;             // [QS] producer -> MMA, compute
  uint64_t* q_empty = q_full + QS;         // [QS] MMA commit (1) + compute warps (8)
  uint64_t* do_full = q_empty + QS;        // [DS]
  uint64_t* do_empty = do_full + DS;       // [DS] MMA commit
  uint64_t* s_full = do_empty + DS;        // MMA -> compute
  uint64_t* p_ready = s_full + 1;          // compute (256) -> MMA
  uint64_t* dp_full = p_ready + 1;         // MMA -> compute
  uint64_t* ds_ready = dp_full + 1;        // compute (256) -> MMA
  uint64_t* ds_free = ds_ready + 1;        // MMA commit -> compute (dS^T image reusable)
  uint64_t* dq_full = ds_free + 1;         // MMA -> drain
  uint64_t* dq_empty = dq_full + 1;        // drain (128) -> MMA
  uint64_t* acc_done = dq_empty + 1;       // MMA -> compute (epilogue)
  uint64_t* acc_free = acc_done + 1;       // compute (256) -> MMA
  uint64_t* it_full = acc_free + 1;        // [kItemRing] work-item ring (sm100.cuh)
  uint64_t* it_empty = it_full + kItemRing;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(it_empty + kItemRing);
  int* sItem = reinterpret_cast<int*>(tmem_slot + 1);      // [kItemRing] (the 16 spare bytes of the layout hold 1 + up to 3; see kSmemBytes)
  const ItemRing ring{sItem, it_full, it_empty};

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    if (smem_u32(smem) & 1023u) __trap();   // tile images need 1024-byte alignment (128B swizzle atoms)
    mbar_init(kv_full, 1); mbar_init(kv_free, 1);
    for (int s = 0; s < QS; ++s) { mbar_init(&q_full[s], 1); mbar_init(&q_empty[s], 9); }
    for (int s = 0; s < DS; ++s) { mbar_init(&do_full[s], 1); mbar_init(&do_empty[s], 1); }
    mbar_init(s_full, 1); mbar_init(p_ready, 256);
    mbar_init(dp_full, 1); mbar_init(ds_ready, 256);
    mbar_init(ds_free, 1);
    mbar_init(dq_full, 1); mbar_init(dq_empty, 128);
    mbar_init(acc_done, 1); mbar_init(acc_free, 256);
    for (int s = 0; s < kItemRing; ++s) { mbar_init(&it_full[s], 1); mbar_init(&it_empty[s], 13); }   // consumers: MMA + 8 compute + 4 drain warps
    fence_mbar_init();
  }
  if (warp == 13) { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
  tc_fence_before();
  __syncthreads();
  if (pd.cta_trace && threadIdx.x == 0) pd.cta_trace[(1 * kTraceMaxCtas + blockIdx.x) * 2] = globaltimer_ns();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const size_t head_stride = static_cast<size_t>(pd.n_tiles_total) * TILE;


  if (warp == 12) {
    // ------------------------------------------------------------------ producer
    setmaxnreg_dec<56>();
    uint32_t it = 0, g = 0;
    for (;; ++it) {
      const int item = item_fetch_producer(ring, it, pd.work_counter + 1, pd.n_items, lane);
      if (item < 0) break;
      const WorkItem wi = pd.dyn_items[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      const size_t hoff = wi.head * head_stride;
      mbar_wait(kv_free, (it & 1) ^ 1);
      {
        const size_t xoff = hoff + static_cast<size_t>(sq.tile_base + wi.tile) * TILE;
        const bool raw = bp.v_raw.base != nullptr;
        const int valid = min(kTileRows, sq.len - wi.tile * kTileRows), tok0 = sq.tok_start + wi.tile * kTileRows;
        const uint32_t vbytes = raw ? raw_tile_stage<D>(sV, bp.v_raw, wi.head, tok0, valid, lane) : TILE;
        if (lane == 0) {
          mbar_expect_tx(kv_full, TILE + vbytes);
          bulk_g2s(sK, bp.kt + xoff, TILE, kv_full);
          if (raw) raw_tile_issue<D>(sV, vmaps, bp.v_raw, wi.head, tok0, valid, kv_full);
          else bulk_g2s(sV, bp.vt + xoff, TILE, kv_full);
        }
      }
      for (int i = 0; i < sq.qt_n; ++i, ++g) {
        const int qt = sq.qt_lo + i;
        const size_t yoff = hoff + static_cast<size_t>(sq.tile_base + qt) * TILE;
        const size_t roff = (static_cast<size_t>(wi.head) * pd.n_tiles_total + sq.tile_base + qt) * kTileRows;
        const uint32_t qs = g % QS, qph = (g / QS) & 1, ds = g % DS, dph = (g / DS) & 1;
        mbar_wait(&q_empty[qs], qph ^ 1);
        if (lane == 0) {
          mbar_expect_tx(&q_full[qs], TILE + 1024);
          bulk_g2s(sQ + qs * TILE, bp.qt + yoff, TILE, &q_full[qs]);
          bulk_g2s(sLse + qs * 128, bp.lse2_t + roff, 512, &q_full[qs]);
          bulk_g2s(sDelta + qs * 128, bp.delta_t + roff, 512, &q_full[qs]);
        }
        mbar_wait(&do_empty[ds], dph ^ 1);
        if (bp.do_raw.base != nullptr) {
          const int valid = min(kTileRows, sq.len - qt * kTileRows), tok0 = sq.tok_start + qt * kTileRows;
          const uint32_t bytes = raw_tile_stage<D>(sdO + ds * TILE, bp.do_raw, wi.head, tok0, valid, lane);
          if (lane == 0) {
            mbar_expect_tx(&do_full[ds], bytes);
            raw_tile_issue<D>(sdO + ds * TILE, domaps, bp.do_raw, wi.head, tok0, valid, &do_full[ds]);
          }
        } else if (lane == 0) {
          mbar_expect_tx(&do_full[ds], TILE);
          bulk_g2s(sdO + ds * TILE, bp.dot + yoff, TILE, &do_full[ds]);
        }
        __syncwarp();
      }
    }
  } else if (warp == 13) {
    // ------------------------------------------------------------------ MMA issuer
    setmaxnreg_dec<56>();
    // Operand formats: S^T is recomputed from the forward's fp16 Q^', K^ images (same bytes -> same logits as
    // the stored LSE was built from); dS^T is fp16 as well (scaled by the group's power of two sk), so that it can pair with
    // those images in dK~ and dQ~; P^T, V and dO stay bf16 (range).
    constexpr uint32_t idesc_s = make_idesc(128, 128, FMT_F16, FMT_F16, MAJOR_K, MAJOR_K);
    constexpr uint32_t idesc_dp = make_idesc(128, 128, FMT_BF16, FMT_BF16, MAJOR_K, MAJOR_K);
    constexpr uint32_t idesc_dv = make_idesc(128, D, FMT_BF16, FMT_BF16, MAJOR_K, MAJOR_MN);
    constexpr uint32_t idesc_dk = make_idesc(128, D, FMT_F16, FMT_F16, MAJOR_K, MAJOR_MN);
    constexpr uint32_t idesc_dq = make_idesc(128, D, FMT_F16, FMT_F16, MAJOR_MN, MAJOR_MN);
    const uint32_t aK = smem_u32(sK), aV = smem_u32(sV), aQ = smem_u32(sQ), adO = smem_u32(sdO), adS = smem_u32(sdS);
    const uint32_t tS = tbase + Cfg::kColS, tdP = tbase + Cfg::kColDP, tdV = tbase + Cfg::kColDV, tdK = tbase + Cfg::kColDK;
    uint32_t it = 0, g0 = 0;
    // S^T of global iteration g
    auto issue_S = [&](uint32_t g) {
      const uint32_t qs = g % QS, qph = (g / QS) & 1;
      mbar_wait(&q_full[qs], qph);
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t koff = (kk >> 2) * BLK + (kk & 3) * 32;
          umma_ss(tS, make_sdesc(aK + koff, 16, 1024), make_sdesc(aQ + qs * TILE + koff, 16, 1024), idesc_s, kk > 0);
        }
        umma_commit(s_full);
      }
      __syncwarp();
    };
    // dP^T of global iteration g (its TMEM columns held dQ~ of iteration g-1)
    auto issue_P = [&](uint32_t g) {
      const uint32_t ds = g % DS, dph = (g / DS) & 1;
      mbar_wait(&do_full[ds], dph);
      if (g > 0) mbar_wait(dq_empty, (g - 1) & 1);
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int kk = 0; kk < D / 16; ++kk) {
          const uint32_t koff = (kk >> 2) * BLK + (kk & 3) * 32;
          umma_ss(tdP, make_sdesc(aV + koff, 16, 1024), make_sdesc(adO + ds * TILE + koff, 16, 1024), idesc_dp, kk > 0);
        }
        umma_commit(dp_full);
      }
      __syncwarp();
    };
    // dV += P^T dO   (P^T bf16 at S columns [0,32) for queries 0-63 and [64,96) for queries 64-127)
    auto issue_V = [&](uint32_t g, bool first) {
      const uint32_t ds = g % DS;
      mbar_wait(p_ready, g & 1);
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t acol = (kk < 4) ? kk * 8 : 64 + (kk - 4) * 8;
          umma_ts(tdV, tS + acol, make_sdesc(adO + ds * TILE + kk * 2048, BLK, 1024), idesc_dv, (!first || kk > 0) ? 1u : 0u);
        }
        umma_commit(&do_empty[ds]);
      }
      __syncwarp();
    };
    // dQ~ = dS K^  and  dK~ += dS^T Q^
    auto issue_QK = [&](uint32_t g, bool first) {
      const uint32_t qs = g % QS;
      mbar_wait(ds_ready, g & 1);
      tc_fence_after();
      if (elect_one()) {
#pragma unroll
        for (int kk = 0; kk < 8; ++kk)
          umma_ss(tdP, make_sdesc(adS + kk * 2048, BLK, 1024), make_sdesc(aK + kk * 2048, BLK, 1024), idesc_dq, kk > 0);
        umma_commit(dq_full);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const uint32_t koff = (kk >> 2) * BLK + (kk & 3) * 32;
          umma_ss(tdK, make_sdesc(adS + koff, 16, 1024), make_sdesc(aQ + qs * TILE + kk * 2048, BLK, 1024), idesc_dk,
                  (!first || kk > 0) ? 1u : 0u);
        }
        umma_commit(&q_empty[qs]);
        umma_commit(ds_free);
      }
      __syncwarp();
    };
    for (;; ++it) {
      const int item = item_fetch_consumer(ring, it, lane);
      if (item < 0) break;
      const WorkItem wi = pd.dyn_items[item];
      const uint32_t n = pd.seqs[wi.seq].qt_n;        // query tiles this process visits (all, unless context-parallel)
      mbar_wait(kv_full, it & 1);
      issue_S(g0);
      issue_P(g0);
      mbar_wait(acc_free, (it & 1) ^ 1);       // previous item's epilogue has drained dV / dK~
      issue_V(g0, true);
      if (n > 1) issue_S(g0 + 1);
      for (uint32_t i = 0; i < n; ++i) {
        issue_QK(g0 + i, i == 0);
        if (i + 1 < n) {
          issue_P(g0 + i + 1);
          issue_V(g0 + i + 1, false);
          if (i + 2 < n) issue_S(g0 + i + 2);
        }
      }
      if (elect_one()) { umma_commit(acc_done); umma_commit(kv_free); }
      __syncwarp();
      g0 += n;
    }
  } else if (warp < 8) {
    // ------------------------------------------------------------------ compute (P^T, dS^T) + epilogue
    const int wg = warp >> 2;                                  // 0: query columns [0,64)   1: [64,128)
    const int r = (warp & 3) * 32 + lane;                      // key row inside the tile == TMEM lane
    const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tS = tbase + Cfg::kColS + lane_base + wg * 64;
    const uint32_t tdP = tbase + Cfg::kColDP + lane_base + wg * 64;
    uint8_t* dS_row = sdS + wg * BLK + r * 128;                // this row's 128 bytes in block wg of the dS^T image
    uint32_t it = 0, g = 0;
    for (;; ++it) {
      const int item = item_fetch_consumer(ring, it, lane);
      if (item < 0) break;
      const WorkItem wi = pd.dyn_items[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      const float2 skv = *reinterpret_cast<const float2*>(pd.grp_sk + (static_cast<size_t>(wi.seq) * pd.H + wi.head) * 4);
      const float sk = skv.x;                    // dS is rounded to fp16 as dS * sk (delta already carries sk: bwd_scale_kernel)
      for (int i = 0; i < sq.qt_n; ++i, ++g) {
        const uint32_t qs = g % QS, qph = (g / QS) & 1;
        const float* lse_s = sLse + qs * 128 + wg * 64;
        const float* dl_s = sDelta + qs * 128 + wg * 64;
        float p[64];
        mbar_wait(&q_full[qs], qph);             // lse2 / delta of this query tile have landed
        mbar_wait(s_full, g & 1);
        tc_fence_after();
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t sv[32];
          tmem_ld32(tS + half * 32, sv);
          tmem_wait_ld();
          uint32_t pk[16];
#pragma unroll
          for (int c = 0; c < 32; c += 4) {
            // lse2 / delta are the same for every thread (broadcast reads): 16-byte loads keep the shared-memory data pipe,
            // which the tensor core's operand reads already load to ~60 %, as free as possible (profiles/r2_ncu.md)
            const float4 l4 = *reinterpret_cast<const float4*>(&lse_s[half * 32 + c]);
            const float p0 = ex2_approx(__uint_as_float(sv[c]) - l4.x);       // S^T is already in the exp2 domain (Q^')
            const float p1 = ex2_approx(__uint_as_float(sv[c + 1]) - l4.y);
            const float p2 = ex2_approx(__uint_as_float(sv[c + 2]) - l4.z);
            const float p3 = ex2_approx(__uint_as_float(sv[c + 3]) - l4.w);
            p[half * 32 + c] = p0; p[half * 32 + c + 1] = p1; p[half * 32 + c + 2] = p2; p[half * 32 + c + 3] = p3;
            pk[c >> 1] = pack_bf16x2(p0, p1);
            pk[(c >> 1) + 1] = pack_bf16x2(p2, p3);
          }
          tmem_st16(tS + half * 16, pk);         // P^T (bf16 pairs) over the already-read S^T columns
        }
        tmem_wait_st();
        tc_fence_before();
        mbar_arrive(p_ready);
        // ---- dS^T = P^T * (dP^T - delta)
        mbar_wait(dp_full, g & 1);
        if (g > 0) mbar_wait(ds_free, (g - 1) & 1);   // dQ~/dK~ GEMMs of the previous tile are done with the image
        tc_fence_after();
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t dpv[32];
          tmem_ld32(tdP + half * 32, dpv);
          tmem_wait_ld();
#pragma unroll
          for (int c8 = 0; c8 < 4; ++c8) {
            uint32_t w[4];
#pragma unroll
            for (int e = 0; e < 8; e += 4) {
              const int c = c8 * 8 + e;
              const float4 d4 = *reinterpret_cast<const float4*>(&dl_s[half * 32 + c]);
              const float ds0 = p[half * 32 + c] * fmaf(__uint_as_float(dpv[c]), sk, -d4.x);
              const float ds1 = p[half * 32 + c + 1] * fmaf(__uint_as_float(dpv[c + 1]), sk, -d4.y);
              const float ds2 = p[half * 32 + c + 2] * fmaf(__uint_as_float(dpv[c + 2]), sk, -d4.z);
              const float ds3 = p[half * 32 + c + 3] * fmaf(__uint_as_float(dpv[c + 3]), sk, -d4.w);
              w[e >> 1] = pack_f16x2(ds0, ds1);
              w[(e >> 1) + 1] = pack_f16x2(ds2, ds3);
            }
            const uint32_t chunk = half * 4 + c8;
            *reinterpret_cast<uint4*>(dS_row + ((chunk ^ (r & 7)) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
          }
        }
        tc_fence_before();
        fence_proxy_async_smem();                // dS^T image -> visible to the tensor core (async proxy)
        mbar_arrive(ds_ready);
        __syncwarp();
        if (lane == 0) mbar_arrive(&q_empty[qs]);   // this warp is done with lse2/delta of the stage
      }
      // ---- epilogue: warps 0-3 store dV (bf16), warps 4-7 store dK~ * scale (fp32)
      mbar_wait(acc_done, it & 1);
      tc_fence_after();
      const int n = wi.tile * kTileRows + r;
      const bool valid_row = n < sq.len;
      const size_t out_off = (static_cast<size_t>(sq.tok_start + n) * pd.H + wi.head) * D;
      const uint32_t tA = tbase + (wg == 0 ? Cfg::kColDV : Cfg::kColDK) + lane_base;
      const bool dv_bf16 = wg == 0 && bp.gv_t == nullptr;      // CP: dV leaves as an fp32 partial like dK~
      // dk~ = scale * dS^T q~ = ln2 * dS^T Q^' (Q^' = q~ * scale * log2e), and dS carries sk
      const float sc = wg == 0 ? 1.0f : 0.6931471805599453f * skv.y;
      float* f32_out = wg == 0 ? bp.gv_t : bp.gk_t;
      __nv_bfloat16* dv_row = (valid_row && dv_bf16) ? raw_row<__nv_bfloat16>(pd.sh, bp.dv, sq.tok_start + n, wi.head, D) : nullptr;
#pragma unroll
      for (int c = 0; c < D / 32; ++c) {
        uint32_t a[32];
        tmem_ld32(tA + c * 32, a);
        tmem_wait_ld();
        if (valid_row) {
          if (dv_bf16) {
#pragma unroll
            for (int i2 = 0; i2 < 32; i2 += 8) {
              uint4 w;
              w.x = pack_bf16x2(__uint_as_float(a[i2]), __uint_as_float(a[i2 + 1]));
              w.y = pack_bf16x2(__uint_as_float(a[i2 + 2]), __uint_as_float(a[i2 + 3]));
              w.z = pack_bf16x2(__uint_as_float(a[i2 + 4]), __uint_as_float(a[i2 + 5]));
              w.w = pack_bf16x2(__uint_as_float(a[i2 + 6]), __uint_as_float(a[i2 + 7]));
              *reinterpret_cast<uint4*>(dv_row + c * 32 + i2) = w;
            }
          } else {
#pragma unroll
            for (int i2 = 0; i2 < 32; i2 += 4) {
              float4 f;
              f.x = __uint_as_float(a[i2]) * sc; f.y = __uint_as_float(a[i2 + 1]) * sc;
              f.z = __uint_as_float(a[i2 + 2]) * sc; f.w = __uint_as_float(a[i2 + 3]) * sc;
              *reinterpret_cast<float4*>(f32_out + out_off + c * 32 + i2) = f;
            }
          }
        }
      }
      tc_fence_before();
      mbar_arrive(acc_free);
    }
  } else if (warp < 12) {
    // ------------------------------------------------------------------ dQ~ drain (warps 8-11)
    setmaxnreg_inc<200>();
    const int q = (warp & 3) * 32 + lane;                      // query row inside the tile == TMEM lane
    const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t tdQ = tbase + Cfg::kColDP + lane_base;
    const bool leader = threadIdx.x == 256;
    float sc = 0.f;                                                 // softmax_scale / sk of the current item (x the row's qs, fixed point)
    float sc_item = 0.f;
    float amax = 0.f;                                               // fixed point: largest |scaled partial| of the current tile (NaN if any was)
    float* stage_row = reinterpret_cast<float*>(sStage) + q * 32;   // row q of staging buffer 0; buffer 1 at +128*32
    uint32_t g = 0;
    // chunk = 32 d-columns of the tile (16 KB, contiguous in the blocked global layout).  Two staging
    // buffers alternate; before a buffer is rewritten, the bulk reduce issued from it two chunks ago
    // must have finished READING it (wait_group.read 1 = all but the most recent group).
    auto flush_chunk = [&](const uint32_t (&v)[32], int chunk, float* gtile) {
      if (leader) bulk_wait_group_read<1>();
      named_bar_sync(1, 128);
      float* dst = stage_row + (chunk & 1) * (kTileRows * 32);
      if (bp.dq_fixed) {
        // fixed point: sc carries the row's qs; round to nearest, |value| <= 2^30 by the bound above (amax checks it: a
        // NaN-propagating maximum, one FMNMX per value)
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float f0 = __uint_as_float(v[4 * j]) * sc, f1 = __uint_as_float(v[4 * j + 1]) * sc;
          const float f2 = __uint_as_float(v[4 * j + 2]) * sc, f3 = __uint_as_float(v[4 * j + 3]) * sc;
          amax = max_nan(max_nan(amax, fabsf(f0)), fabsf(f1));
          amax = max_nan(max_nan(amax, fabsf(f2)), fabsf(f3));
          int4 q4;
          q4.x = __float2int_rn(f0); q4.y = __float2int_rn(f1); q4.z = __float2int_rn(f2); q4.w = __float2int_rn(f3);
          *reinterpret_cast<int4*>(dst + ((j ^ (q & 7)) << 2)) = q4;
        }
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          float4 f;
          f.x = __uint_as_float(v[4 * j]) * sc; f.y = __uint_as_float(v[4 * j + 1]) * sc;
          f.z = __uint_as_float(v[4 * j + 2]) * sc; f.w = __uint_as_float(v[4 * j + 3]) * sc;
          *reinterpret_cast<float4*>(dst + ((j ^ (q & 7)) << 2)) = f;
        }
      }
      fence_proxy_async_smem();
      named_bar_sync(1, 128);
      if (leader) {
        void* g = gtile + chunk * (kTileRows * 32);
        const void* src = sStage + (chunk & 1) * (kTileRows * 32 * 4);
        if (bp.dq_fixed) bulk_reduce_add_s32_s2g(g, src, kTileRows * 32 * 4);
        else bulk_reduce_add_f32_s2g(g, src, kTileRows * 32 * 4);
        bulk_commit_group();
      }
    };
    for (uint32_t it = 0;; ++it) {
      const int item = item_fetch_consumer(ring, it, lane);
      if (item < 0) break;
      const WorkItem wi = pd.dyn_items[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      {
        // dq~ = softmax_scale * dS k~, dS carries sk; fixed-point mode: times the query row's power of two qs_i (bwd_scale_kernel)
        const float2 gs = *reinterpret_cast<const float2*>(pd.grp_sk + (static_cast<size_t>(wi.seq) * pd.H + wi.head) * 4);
        sc = sc_item = pd.softmax_scale * gs.y;
      }
      for (int i = 0; i < sq.qt_n; ++i, ++g) {
        const int qt = sq.qt_lo + i;
        const size_t tile_idx = static_cast<size_t>(wi.head) * pd.n_tiles_total + sq.tile_base + qt;
        float* gtile = bp.gq_blk + tile_idx * (kTileRows * D);
        float* row_qs = bp.rowqs_t + tile_idx * kTileRows + q;       // (dereferenced in fixed-point mode only)
        if (bp.dq_fixed) { sc = sc_item * *row_qs; amax = 0.f; }
        mbar_wait(dq_full, g & 1);
        tc_fence_after();
        uint32_t v0[32], v1[32];
        tmem_ld32(tdQ, v0);
        tmem_ld32(tdQ + 32, v1);
        tmem_wait_ld();
        if constexpr (D == 64) { tc_fence_before(); mbar_arrive(dq_empty); }
        flush_chunk(v0, 0, gtile);
        flush_chunk(v1, 1, gtile);
        if constexpr (D == 128) {
          tmem_ld32(tdQ + 64, v0);
          tmem_ld32(tdQ + 96, v1);
          tmem_wait_ld();
          tc_fence_before();
          mbar_arrive(dq_empty);                 // dQ~ columns are free for the next dP^T
          flush_chunk(v0, 2, gtile);
          flush_chunk(v1, 3, gtile);
        }
        // All writers of a row's mark store the same value and a concurrent reader that picks it up produces NaN partials
        // (-> 0 after cvt) and marks the row again: the row's dQ is NaN either way.
        if (bp.dq_fixed && !(amax <= 1073741824.0f)) *row_qs = __int_as_float(0x7fc00000);
      }
    }
    if (leader) bulk_wait_group<0>();            // all reductions have been performed before the CTA exits
  } else {
    setmaxnreg_dec<56>();                        // warps 14-15: only there to complete the fourth warpgroup
  }
  tc_fence_before();
  __syncthreads();
  if (pd.cta_trace && threadIdx.x == 0) pd.cta_trace[(1 * kTraceMaxCtas + blockIdx.x) * 2 + 1] = globaltimer_ns();
  if (warp == 13) tmem_dealloc(tbase, 512);
}

}  // namespace arachne
