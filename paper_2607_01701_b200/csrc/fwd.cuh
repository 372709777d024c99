// Forward kernel (§8 a2-a4): persistent, warp-specialised, tcgen05 + TMEM, two query tiles in flight.
//
// Work item = (sequence b, head h, PAIR of 128-row query tiles) (a trailing odd tile runs alone).
// Items are taken DYNAMICALLY from the plan's LPT-ordered list: lane 0 of the producer warp does an atomicAdd on a per-launch
// counter and hands the index to the other warp roles through a 4-slot shared-memory ring (sm100.cuh, ItemRing).
// Per item the CTA streams the ceil(L_b/128) key/value tiles of sequence b ONLY (block-diagonal:
// no other tile is ever touched, no masked-out tile is computed).  The two query tiles ping-pong on
// the tensor pipe so that the softmax of one overlaps the GEMMs of the other:
//
//   issue order   S0_0 S1_0 | PV0_0 S0_1 PV1_0 S1_1 | PV0_1 S0_2 PV1_1 S1_2 | ...
//
//   warp 8  producer : Q^ images (cp.async.bulk), then K^_j (cp.async.bulk of the image) and V_j (tensor-map TMA straight from
//                      the caller's tensor, rawtile.cuh; an image only for sharded plans) into a ring of tile slots
//   warp 9  MMA      : S_t,j = Q^_t K^_j^T  (SS, fp16 x fp16 -> fp32 TMEM, one buffer per query tile)
//                      O_t  += P_t,j V_j    (TS: P bf16 in TMEM aliasing S_t; V MN-major)
//   warps 0-3 / 4-7  : softmax of query tile 0 / 1, one query row per thread: tcgen05.ld S row, exp2, P -> bf16 -> tcgen05.st,
//                      handed to the MMA warp in two halves of 64 keys (kSplitP) so that PV of the first half runs under the
//                      exponentiation of the second; final O / l -> bf16, LSE -> fp32.  QK-RMSNorm bounds the logits, so the
//                      default is a STATIC max (p = 2^s, no running max, no rescale); unbounded logits (no_norm, huge gamma)
//                      take online softmax with LAZY rescaling (O only rescaled when a row max grew by > 2^8).
// Forms: fwd_kernel (one CTA per item; <D, true> = fused Q, the in-kernel A/B of §8 a1), fwd_pair_kernel (cluster of 2,
// cta_group::2 MMAs), fwd_mc_kernel (cluster of 2 sharing the K^/V stream by TMA multicast).
//
// Q^, K^ are fp16 (RMSNorm bounds |x^_d| <= gamma_max * sqrt(D)); fp16 operands put the LSE
// error floor at ~2e-4 instead of ~1.5e-3 for bf16.  P and V are bf16.
#pragma once
#include "common.cuh"
#include "normrope.cuh"
#include "rawtile.cuh"
#include "sm100.cuh"

namespace arachne {

struct FwdParams {
  const uint8_t* qt;      // [H][n_tiles][TILE_BYTES]  Q^ fp16 images
  const uint8_t* kt;      // K^ fp16 images
  const uint8_t* vt;      // V bf16 images (only when v_raw.base == nullptr)
  RawTensor v_raw;        // base != nullptr: V tiles come straight from the raw tensor by tensor-map TMA (rawtile.cuh)
  RawTensor q_raw;        // base != nullptr (ARACHNE_FLAG_FWD_FUSED_Q, one-CTA form): the item's RAW query tiles are loaded by
                          // tensor-map TMA and normalised + rotated + rounded to fp16 in place by the softmax warps ("fused into
                          // the Q load" in the literal sense; the A/B partner of the prologue)
  const float* gamma_q;   // fused Q only
  float q_prescale;       // fused Q only: softmax_scale * log2(e)
  ShardedPtr o;           // [N,H_total,D] bf16, possibly sharded by token range (common.cuh)
  float* lse;             // [H,N]
  unsigned* envelope;     // plan-owned sticky word: float bits of the largest logit bound that exceeded bound_limit
  float bound_limit;      // logit bound (log2 units) the gates are claimed for; +inf with ARACHNE_FLAG_WIDE_LOGITS
};

// A/B switches (profiles/r2_fwd_handoff.md).  kSplitP = number of pieces (1, 2 or 4) in which the softmax hands a tile of P to
// the MMA warp: with more than one, the first pieces of O += P V run on the tensor pipe while the rest of the row is still
// being exponentiated (the MUFU time of a tile, 1024 clk, is as long as its two GEMMs; every cycle of the
// S -> exp -> PV -> S chain that is not overlapped is lost on both units).  kWarpArrive: one mbarrier arrival per softmax
// WARP (after __syncwarp) instead of one per thread.
#ifndef ARACHNE_FWD_SPLIT_P
#define ARACHNE_FWD_SPLIT_P 2
#endif
#ifndef ARACHNE_FWD_WARP_ARRIVE
#define ARACHNE_FWD_WARP_ARRIVE 0
#endif
constexpr int kSplitP = ARACHNE_FWD_SPLIT_P;
static_assert(kSplitP == 1 || kSplitP == 2 || kSplitP == 4, "P is handed over in 1, 2 or 4 pieces of 128 / kSplitP keys");
constexpr bool kWarpArrive = ARACHNE_FWD_WARP_ARRIVE != 0;

// kPair = true: the CTA-PAIR form of the kernel (cluster of 2, tcgen05 cta_group::2; D = 128 only).  A pair takes items of up
// to FOUR query tiles — CTA r of the pair owns tiles 2r, 2r+1 of the item — and shares every K^/V tile: each CTA loads and
// holds only HALF of it (K^: its 64 keys x D; V: all 128 keys x its 64 d-columns), the leader CTA's MMA warp issues M = 256
// instructions that cover the same-numbered query tile of both CTAs, and completion is multicast to the barriers of both.
// Per SM this halves the K/V traffic from L2 and the B-operand reads from shared memory (the S GEMM, both operands in shared
// memory, is otherwise pinned at the 128 B/clk shared-memory limit: DESIGN.md §7).  The peer CTA's warp 9 has no MMAs to
// issue; it relays "my half has landed" to the leader.  Softmax / epilogue warps are the same code in both forms.
// kMode 2: the MULTICAST form (cluster of 2, D = 128).  The two CTAs of a cluster are two ordinary one-CTA kernels (their own
// cta_group::1 MMAs, softmax and barriers) that work on the same (sequence, head) — the same 4-tile items as the pair form — and
// SHARE THE K^/V STREAM: each CTA fetches half of every tile and multicasts it into both CTAs' ring slots, so the L2 -> SM
// traffic of the pair halves (profiles/r2_fwd_handoff.md: the loop is sensitive to it).  A slot is refilled once BOTH CTAs'
// tensor cores are done with it (the releasing commits are multicast too: kv_empty counts 2).
enum : int { kFwdSingle = 0, kFwdPair = 1, kFwdMcast = 2 };
template <int D, int kMode = kFwdSingle>
struct FwdCfg {
  static constexpr bool kPair = kMode == kFwdPair;
  static_assert(kMode == kFwdSingle || D == 128, "the CTA-pair forward is built for head_dim 128 (V's d-halves must be whole 128-byte swizzle blocks)");
  static constexpr int kTileBytes = kTileRows * D * 2;
  static constexpr int kSlotBytes = kPair ? kTileBytes / 2 : kTileBytes;   // one ring slot: a K^ or V tile (pair: this CTA's half)
  static constexpr int kRing = kPair ? 8 : ((D == 128) ? 5 : 8);           // K/V ring slots (K_j, V_j alternate)
  static constexpr int kNumBars = 3 + 2 * kRing + 8 + 2 * (kSplitP - 1) + 2 * kItemRing + (kPair ? 1 + kRing : 0);
  static constexpr int kSmemBytes = 2 * kTileBytes + kRing * kSlotBytes + 8 * kNumBars + 16 + 4 * kItemRing;
  static constexpr int kThreads = 320;
  // every other PAIR of exp2 on the FMA pipe (ex2_poly3_x2: packed FADD2 / FFMA2, 4 issue slots per element) instead of MUFU:
  // pays at D = 64, where MUFU (16 ex2/clk/SM) is the busiest unit (cogvideox fwd 12.6 ms vs 12.9 with every 4th exp2 as a scalar
  // polynomial, 14.7 all-MUFU); at D = 128 every variant — scalar or packed, 1/16 to all — is SLOWER than all-MUFU (720p fwd
  // 147.9 / 153.2 / 156.1 / 162.3 ms for 0 / 1/4 / 1/2 / all packed): the softmax warps are bound by their own in-order
  // instruction stream, not by the MUFU pipe (profiles/r2_fwd_handoff.md)
  static constexpr bool kPolyExp = (D == 64);
  // TMEM columns: S0 [0,128) S1 [128,256) O0 [256,256+D) O1 [256+D,256+2D)
  static constexpr uint32_t kColS = 0, kColO = 256;
};

// largest logit bound (log2 units) for which the forward takes the static-max softmax
constexpr float kStaticMaxBound = 32.0f;

// Fused Q (ARACHNE_FLAG_FWD_FUSED_Q): one thread turns one RAW bf16 query row of a tile in shared memory into the fp16 operand
// row, in place: RMSNorm -> 3D RoPE -> x softmax_scale*log2(e) -> fp16, with the prologue's arithmetic in the prologue's order
// (normrope.cuh; the chunk sums of squares are combined like prep_kernel's lane butterfly), so the bytes equal the Q^ image's.
// Rows past the sequence end were zeroed by the producer and stay zero.
template <int D>
__device__ __forceinline__ void fused_q_row(const ProblemDesc& pd, const FwdParams& fp, uint8_t* tile, const SeqInfo& sq, int n, int row) {
  constexpr int NCH = D / 8;
  if (n >= sq.len) return;
  const TokInfo ti = pd.tok_info[sq.tok_start + n];
  const bool rotate = !pd.no_rope && !(ti.t_flag >> 31);
  float rinv = 1.0f;
  if (!pd.no_norm) {
    float c[NCH];
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
      float x[8];
      unpack_bf16x8(*reinterpret_cast<const uint4*>(tile + image_off(row, ch * 8)), x);
      c[ch] = sumsq8(x);
    }
#pragma unroll
    for (int o = NCH / 2; o > 0; o >>= 1)
#pragma unroll
      for (int j = 0; j < NCH; ++j)
        if ((j & o) == 0) { const float sum = c[j] + c[j ^ o]; c[j] = sum; c[j ^ o] = sum; }
    rinv = rsqrtf(c[0] * (1.0f / D) + pd.eps);
  }
#pragma unroll 2
  for (int ch = 0; ch < NCH; ++ch) {
    uint4* p = reinterpret_cast<uint4*>(tile + image_off(row, ch * 8));
    float x[8], gam[8];
    unpack_bf16x8(*p, x);
#pragma unroll
    for (int i = 0; i < 8; ++i) gam[i] = fp.gamma_q ? __ldg(&fp.gamma_q[ch * 8 + i]) : 1.0f;
    float2 cs[4];
    rope_cs4(pd.rope, ch * 8, ti, rotate, cs);
    norm_rope_apply8(x, gam, cs, pd.no_norm != 0, rinv, fp.q_prescale);
    *p = pack8(x, FMT_F16);
  }
}

template <int D, int kMode, bool kFusedQ = false>
__device__ __forceinline__ void fwd_body(const ProblemDesc& pd, const FwdParams& fp, const RawMaps& vm, const RawMaps& qm) {
  using Cfg = FwdCfg<D, kMode>;
  constexpr bool kPair = kMode == kFwdPair;      // cta_group::2 MMAs issued by the leader for both CTAs
  constexpr bool kMc = kMode == kFwdMcast;       // independent CTAs sharing the K^/V stream by multicast
  constexpr bool kCl = kMode != kFwdSingle;      // any cluster form: 4-tile items handed out by the leader
  constexpr int TILE = Cfg::kTileBytes;
  constexpr int SLOT = Cfg::kSlotBytes;
  constexpr int RING = Cfg::kRing;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* sQ = smem;                     // 2 tiles
  uint8_t* sKV = sQ + 2 * TILE;           // RING slots
  uint64_t* bars = reinterpret_cast<uint64_t*>(sKV + RING * SLOT);
  uint64_t* q_full = bars;            // producer -> MMA
  uint64_t* q_empty = bars + 1;       // MMA (commit) -> producer
  uint64_t* q_ready = bars + 2;       // fused Q: softmax warps (256 arrivals) -> MMA: the Q^ tiles have been normalised in place
  uint64_t* kv_full = bars + 3;       // [RING]
  uint64_t* kv_empty = kv_full + RING;
  uint64_t* s_full = kv_empty + RING;    // [2] MMA (commit) -> softmax of tile t
  uint64_t* p_full = s_full + 2;         // [2] softmax (128 arrivals) -> MMA
  uint64_t* pa_full = p_full + 2;        // [2][kSplitP - 1] softmax -> MMA: piece i of P (keys [i, i+1) * 128 / kSplitP) is in TMEM
  uint64_t* pv_done = pa_full + 2 * (kSplitP - 1);   // [2] MMA (commit) -> softmax: one phase per PV
  uint64_t* o_free = pv_done + 2;        // [2] softmax epilogue (128 arrivals) -> MMA
  uint64_t* it_full = o_free + 2;        // [kItemRing] work-item ring (sm100.cuh): items are taken dynamically
  uint64_t* it_empty = it_full + kItemRing;
  uint64_t* peer_q_full = it_empty + kItemRing;        // pair, LEADER only: the peer's Q^ tiles / K,V halves have landed
  uint64_t* peer_kv_full = peer_q_full + 1;            //   [RING]  (arrived remotely by the peer's relay warp)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(it_empty + kItemRing + (kPair ? 1 + RING : 0));
  int* sItem = reinterpret_cast<int*>(tmem_slot + 1);
  const ItemRing item_ring{sItem, it_full, it_empty};

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = kCl ? cluster_ctarank() : 0u;      // 0 = leader (issues the MMAs, owns the barriers the MMA warp waits on)
  // arrivals of the softmax / epilogue warps on a barrier the MMA warp waits on: 1-CTA form = every thread arrives (count 128);
  // pair form = one arrival per warp on the LEADER's barrier (count 4 local + 4 remote warps)
  constexpr uint32_t kArrivals = kPair ? 8 : (kWarpArrive ? 4 : 128);
  if (threadIdx.x == 0) {
    if (smem_u32(smem) & 1023u) __trap();   // tile images need 1024-byte alignment (128B swizzle atoms)
    mbar_init(q_full, 1); mbar_init(q_empty, 1); mbar_init(q_ready, 256);
    for (int s = 0; s < RING; ++s) { mbar_init(&kv_full[s], 1); mbar_init(&kv_empty[s], kMc ? 2 : 1); }
    for (int t = 0; t < 2; ++t) {
      mbar_init(&s_full[t], 1); mbar_init(&p_full[t], kArrivals);
      for (int i = 0; i < kSplitP - 1; ++i) mbar_init(&pa_full[t * (kSplitP - 1) + i], kArrivals);
      mbar_init(&pv_done[t], 1); mbar_init(&o_free[t], kArrivals);
    }
    // item ring consumers: MMA + 8 softmax warps; pair: + the peer's producer, relay and 8 softmax warps (remote arrivals)
    for (int s = 0; s < kItemRing; ++s) { mbar_init(&it_full[s], 1); mbar_init(&it_empty[s], kCl ? 19 : 9); }
    if constexpr (kPair) {
      mbar_init(peer_q_full, 1);
      for (int s = 0; s < RING; ++s) mbar_init(&peer_kv_full[s], 1);
    }
    fence_mbar_init();
  }
  if (warp == 9) {
    if constexpr (kPair) { tmem_alloc2(tmem_slot, 512); tmem_relinquish2(); }
    else { tmem_alloc(tmem_slot, 512); tmem_relinquish(); }
  }
  tc_fence_before();
  if constexpr (kCl) cluster_sync_all(); else __syncthreads();      // (cluster: barrier inits visible to the peer's remote arrivals)
  if (pd.cta_trace && threadIdx.x == 0) pd.cta_trace[(0 * kTraceMaxCtas + blockIdx.x) * 2] = globaltimer_ns();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;
  const size_t head_stride = static_cast<size_t>(pd.n_tiles_total) * TILE;
  const WorkItem* item_list = kCl ? pd.dyn_fwd_pair_items : pd.dyn_fwd_items;
  const int n_list = kCl ? pd.n_fwd_pair_items : pd.n_fwd_items;
  auto wait = [](uint64_t* bar, uint32_t parity) { if constexpr (kCl) mbar_wait_wd(bar, parity); else mbar_wait(bar, parity); };
  // item hand-out.  1-CTA: sm100.cuh ItemRing.  Pair: the LEADER's producer takes the index and publishes it to both CTAs'
  // rings; every consumer warp of both CTAs releases the slot on the LEADER's `empty` barrier.
  auto fetch_producer = [&](uint32_t it) -> int {
    if constexpr (!kCl) return item_fetch_producer(item_ring, it, pd.work_counter, n_list, lane);
    const uint32_t s = it % kItemRing, ph = (it / kItemRing) & 1;
    int item = 0;
    if (lane == 0) {
      mbar_wait_wd(&it_empty[s], ph ^ 1);
      item = atomicAdd(pd.work_counter, 1);
      if (item >= n_list) item = -1;
      sItem[s] = item;
      st_cluster_u32(mapa_u32(smem_u32(&sItem[s]), 1), static_cast<uint32_t>(item));
      mbar_arrive(&it_full[s]);
      mbar_arrive_cluster(mapa_u32(smem_u32(&it_full[s]), 1));     // release.cluster: the peer sees the slot write
    }
    return __shfl_sync(0xffffffffu, item, 0);
  };
  auto fetch_consumer = [&](uint32_t it) -> int {
    if constexpr (!kCl) return item_fetch_consumer(item_ring, it, lane);
    const uint32_t s = it % kItemRing, ph = (it / kItemRing) & 1;
    mbar_wait_wd(&it_full[s], ph);
    const int item = sItem[s];
    __syncwarp();
    if (lane == 0) mbar_arrive_cluster(mapa_u32(smem_u32(&it_empty[s]), 0));
    return item;
  };
  // number of query tiles each CTA works on in this item (pair: both CTAs run the same count; tiles beyond the item's
  // last one are PHANTOMS — a copy of the last real tile whose rows are never stored — because an M = 256 instruction always
  // covers both CTAs)
  auto tiles_per_cta = [](const WorkItem& wi) { return kCl ? min(2, wi.pad) : wi.pad; };

  if (warp == 8) {
    // ------------------------------------------------------------------ producer
    if (blockIdx.x == 0 && lane == 0) {
      // outside the envelope the gates are claimed for (DESIGN.md §6 / R19): leave a sticky mark (arachne_plan_logit_status)
      const float bound = sqrtf(__uint_as_float(pd.stats[0])) * sqrtf(__uint_as_float(pd.stats[1]));
      if (bound > fp.bound_limit) atomicMax(fp.envelope, __float_as_uint(bound));
    }
    uint32_t it = 0, ring = 0;
    for (;; ++it) {
      const int item = (rank == 0) ? fetch_producer(it) : fetch_consumer(it);
      if (item < 0) break;
      const WorkItem wi = item_list[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      const int n_q = tiles_per_cta(wi);
      const uint8_t* hbase_q = fp.qt + wi.head * head_stride;
      const uint8_t* hbase_k = fp.kt + wi.head * head_stride;
      const uint8_t* hbase_v = fp.vt + wi.head * head_stride;
      wait(q_empty, (it & 1) ^ 1);
      bool q_is_raw = false;
      if constexpr (kFusedQ) {
        {      // fused Q: RAW query tiles (rawtile.cuh); the softmax warps normalise them in place
          q_is_raw = true;
          uint32_t bytes = 0;
          for (int t = 0; t < n_q; ++t) {
            const int n0 = (wi.tile + t) * kTileRows;
            bytes += raw_tile_stage<D>(sQ + t * TILE, fp.q_raw, wi.head, sq.tok_start + n0, min(kTileRows, sq.len - n0), lane);
          }
          if (lane == 0) {
            mbar_expect_tx(q_full, bytes);
            for (int t = 0; t < n_q; ++t) {
              const int n0 = (wi.tile + t) * kTileRows;
              raw_tile_issue<D>(sQ + t * TILE, qm, fp.q_raw, wi.head, sq.tok_start + n0, min(kTileRows, sq.len - n0), q_full);
            }
          }
        }
      }
      if (!q_is_raw && lane == 0) {
        mbar_expect_tx(q_full, n_q * TILE);
        if constexpr (!kCl) {
          bulk_g2s(sQ, hbase_q + static_cast<size_t>(sq.tile_base + wi.tile) * TILE, n_q * TILE, q_full);
        } else {
          for (int t = 0; t < n_q; ++t) {      // this CTA's tiles 2*rank + t of the item; phantoms read the item's last tile
            const int qt = wi.tile + min(static_cast<int>(2 * rank) + t, wi.pad - 1);
            bulk_g2s(sQ + t * TILE, hbase_q + static_cast<size_t>(sq.tile_base + qt) * TILE, TILE, q_full);
          }
        }
      }
      for (int j = 0; j < sq.n_tiles; ++j) {
        const size_t off = static_cast<size_t>(sq.tile_base + j) * TILE;
#pragma unroll
        for (int kv = 0; kv < 2; ++kv, ++ring) {
          const uint32_t st = ring % RING, ph = (ring / RING) & 1;
          wait(&kv_empty[st], ph ^ 1);
          if constexpr (!kPair) {
            if (kv == 1 && fp.v_raw.base != nullptr) {      // V_j straight from the raw tensor (rawtile.cuh)
              const int valid = min(kTileRows, sq.len - j * kTileRows);
              const int tok0 = sq.tok_start + j * kTileRows;
              const uint32_t bytes = raw_tile_stage<D>(sKV + st * SLOT, fp.v_raw, wi.head, tok0, valid, lane);
              if (lane == 0) {
                mbar_expect_tx(&kv_full[st], bytes);
                if constexpr (kMc) raw_tile_issue_mc<D>(sKV + st * SLOT, vm, fp.v_raw, wi.head, tok0, valid, &kv_full[st], rank);
                else raw_tile_issue<D>(sKV + st * SLOT, vm, fp.v_raw, wi.head, tok0, valid, &kv_full[st]);
              }
              continue;
            }
          }
          if (lane == 0) {
            mbar_expect_tx(&kv_full[st], SLOT);
            if constexpr (kMc) {
              // this CTA's half of the tile image, into BOTH CTAs' slots
              bulk_g2s_mc(sKV + st * SLOT + rank * (TILE / 2), (kv == 0 ? hbase_k : hbase_v) + off + rank * (TILE / 2), TILE / 2,
                          &kv_full[st], 3);
            } else if constexpr (!kPair) {
              bulk_g2s(sKV + st * SLOT, (kv == 0 ? hbase_k : hbase_v) + off, TILE, &kv_full[st]);
            } else if (kv == 0) {
              // K^: this CTA's 64 keys (rows 64*rank..) of each 64-element block -> [D/64][64 rows][128 B]
#pragma unroll
              for (int c = 0; c < D / 64; ++c)
                bulk_g2s(sKV + st * SLOT + c * 8192, hbase_k + off + c * (kTileRows * 128) + rank * 8192, 8192, &kv_full[st]);
            } else {
              // V: all 128 keys, this CTA's 64 d-columns = block `rank` of the image (contiguous)
              bulk_g2s(sKV + st * SLOT, hbase_v + off + rank * (kTileRows * 128), kTileRows * 128, &kv_full[st]);
            }
          }
        }
        __syncwarp();
      }
    }
  } else if (warp == 9 && kPair && rank != 0) {
    // ------------------------------------------------------------------ pair form, peer CTA: relay "my half has landed"
    if constexpr (kPair) {
      uint32_t it = 0, ring = 0;
      for (;; ++it) {
        const int item = fetch_consumer(it);
        if (item < 0) break;
        const int n_kv = pd.seqs[item_list[item].seq].n_tiles;
        mbar_wait_wd(q_full, it & 1);
        if (lane == 0) mbar_arrive_cluster(mapa_u32(smem_u32(peer_q_full), 0));
        for (int s2 = 0; s2 < 2 * n_kv; ++s2, ++ring) {
          const uint32_t st = ring % RING, ph = (ring / RING) & 1;
          mbar_wait_wd(&kv_full[st], ph);
          if (lane == 0) mbar_arrive_cluster(mapa_u32(smem_u32(&peer_kv_full[st]), 0));
        }
      }
    }
  } else if (warp == 9) {
    // ------------------------------------------------------------------ MMA issuer
    // The whole warp runs the loop convergently (uniform descriptors -> plain UTCHMMA issue, no
    // per-instruction election loop); one elected lane issues the tcgen05 instructions.
    constexpr uint32_t M = kPair ? 256 : 128;
    constexpr uint32_t idesc_s = make_idesc(M, 128, FMT_F16, FMT_F16, MAJOR_K, MAJOR_K);
    constexpr uint32_t idesc_o = make_idesc(M, D, FMT_BF16, FMT_BF16, MAJOR_K, MAJOR_MN);
    constexpr uint32_t KBLK = kPair ? 64 * 128 : kTileRows * 128;     // bytes of one 64-element block of a K^ slot
    const uint32_t aQ = smem_u32(sQ), aKV = smem_u32(sKV);
    auto mma_ss = [](uint32_t d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t acc) { if constexpr (kPair) umma_ss2(d, a, b, idesc, acc); else umma_ss(d, a, b, idesc, acc); };
    auto mma_ts = [](uint32_t d, uint32_t a, uint64_t b, uint32_t idesc, uint32_t acc) { if constexpr (kPair) umma_ts2(d, a, b, idesc, acc); else umma_ts(d, a, b, idesc, acc); };
    auto commit = [](uint64_t* bar) { if constexpr (kPair) umma_commit2(bar); else umma_commit(bar); };
    // releasing a K/V ring slot: in the multicast form the slot is written by BOTH CTAs' producers, so both must hear it
    auto commit_slot = [&](uint64_t* bar) { if constexpr (kMc) umma_commit_mc(bar, 3); else commit(bar); };
    uint32_t it = 0, ring = 0;      // ring: slot counter at K_0 of the current item (K_j = ring+2j, V_j = ring+2j+1)
    uint32_t cnt[2] = {0, 0};       // per query tile: number of PV tiles issued so far
    for (;; ++it) {
      const int item = fetch_consumer(it);
      if (item < 0) break;
      const WorkItem wi = item_list[item];
      const int n_kv = pd.seqs[wi.seq].n_tiles;
      const int n_q = tiles_per_cta(wi);
      // S_t,j : waits K_j on first use, releases the slot (and Q^ after the last tile) on last use
      auto issue_s = [&](int t, int j) {
        const uint32_t r = ring + 2 * j, st = r % RING, ph = (r / RING) & 1;
        if (t == 0) { wait(&kv_full[st], ph); if constexpr (kPair) mbar_wait_wd(&peer_kv_full[st], ph); }
        tc_fence_after();
        if (elect_one()) {
          const uint32_t tS = tbase + Cfg::kColS + t * 128;
#pragma unroll
          for (int kk = 0; kk < D / 16; ++kk) {
            const uint32_t koff = (kk >> 2) * (kTileRows * 128) + (kk & 3) * 32;
            const uint32_t boff = (kk >> 2) * KBLK + (kk & 3) * 32;
            mma_ss(tS, make_sdesc(aQ + t * TILE + koff, 16, 1024), make_sdesc(aKV + st * SLOT + boff, 16, 1024), idesc_s, kk > 0);
          }
          commit(&s_full[t]);
          if (t == n_q - 1) {
            commit_slot(&kv_empty[st]);
            if (j == n_kv - 1) commit(q_empty);
          }
        }
        __syncwarp();
      };
      auto issue_pv = [&](int t, int j) {
        const uint32_t r = ring + 2 * j + 1, st = r % RING, ph = (r / RING) & 1;
        if (t == 0) { wait(&kv_full[st], ph); if constexpr (kPair) mbar_wait_wd(&peer_kv_full[st], ph); }
        if (j == 0) wait(&o_free[t], (it & 1) ^ 1);        // previous item's epilogue has drained O_t
        const uint32_t tP = tbase + Cfg::kColS + t * 128, tO = tbase + Cfg::kColO + t * D;
        constexpr int KPP = (kTileRows / 16) / kSplitP;          // K = 16 steps per piece
#pragma unroll
        for (int piece = 0; piece < kSplitP; ++piece) {
          // pieces before the last: those keys of P have been stored; their share of O += P V runs while the softmax
          // finishes the row
          wait(piece < kSplitP - 1 ? &pa_full[t * (kSplitP - 1) + piece] : &p_full[t], cnt[t] & 1);
          tc_fence_after();
          if (elect_one()) {
#pragma unroll
            for (int kk = piece * KPP; kk < (piece + 1) * KPP; ++kk)
              mma_ts(tO, tP + kk * 8, make_sdesc(aKV + st * SLOT + kk * 2048, kTileRows * 128, 1024), idesc_o, (j > 0 || kk > 0) ? 1u : 0u);
            if (piece == kSplitP - 1) {
              commit(&pv_done[t]);
              if (t == n_q - 1) commit_slot(&kv_empty[st]);
            }
          }
          __syncwarp();
        }
        ++cnt[t];
      };
      wait(q_full, it & 1);
      if constexpr (kFusedQ) wait(q_ready, it & 1);      // fused Q: tiles normalised in place
      if constexpr (kPair) mbar_wait_wd(peer_q_full, it & 1);
      for (int t = 0; t < n_q; ++t) issue_s(t, 0);
      for (int j = 0; j < n_kv; ++j) {
        for (int t = 0; t < n_q; ++t) {
          issue_pv(t, j);
          if (j + 1 < n_kv) issue_s(t, j + 1);
        }
      }
      ring += 2 * n_kv;
    }
  } else {
    // ------------------------------------------------------------------ softmax + epilogue (warps 0-7)
    const int t = warp >> 2;                                              // query tile of the pair
    const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;   // this warp's TMEM lanes
    const uint32_t tS = tbase + Cfg::kColS + t * 128 + lane_base;
    const uint32_t tO = tbase + Cfg::kColO + t * D + lane_base;
    const int row = (warp & 3) * 32 + lane;   // query row inside the tile
    uint32_t g = 0;                // S/PV tile counter of this query tile (matches the MMA warp's cnt[t])
    uint32_t it = 0;
    // Logit bound from the prep kernel: |s'| <= |q~'| |k~| (Cauchy-Schwarz; q~' carries scale*log2e).
    // QK-RMSNorm makes it sqrt(D)*log2(e)*|gamma_q|_inf*|gamma_k|_inf (16.3 for D = 128, gamma = 1), so
    // exp2(s') can be taken with NO running max: p <= 2^32, l <= 2^18 * 2^32, all far inside fp32 / bf16
    // range.  Anything larger (no_norm debug flag, huge gamma) takes the online-softmax path below.
    const float bound = sqrtf(__uint_as_float(pd.stats[0])) * sqrtf(__uint_as_float(pd.stats[1]));
    const bool static_max = bound <= kStaticMaxBound;     // false for NaN / inf
    // arrival on a barrier the MMA warp waits on, after this thread's TMEM traffic has been fenced
    auto arrive_mma = [&](uint64_t* bar) {
      if constexpr (kPair) { __syncwarp(); if (lane == 0) mbar_arrive_cluster(mapa_u32(smem_u32(bar), 0)); }
      else if constexpr (kWarpArrive) { __syncwarp(); if (lane == 0) mbar_arrive(bar); }
      else { mbar_arrive(bar); }
    };
    for (;; ++it) {
      const int item = fetch_consumer(it);
      if (item < 0) break;
      const WorkItem wi = item_list[item];
      const SeqInfo sq = pd.seqs[wi.seq];
      if constexpr (kFusedQ) {
        {      // fused Q: normalise this thread's row of the raw tile in place, then release the MMA warp
          wait(q_full, it & 1);
          if (t < tiles_per_cta(wi)) fused_q_row<D>(pd, fp, sQ + t * TILE, sq, (wi.tile + t) * kTileRows + row, row);
          fence_proxy_async_smem();
          mbar_arrive(q_ready);
        }
      }
      if (t >= tiles_per_cta(wi)) {
        // odd trailing tile: warps 4-7 sit this item out, but keep the o_free phase in step with `it`
        arrive_mma(&o_free[t]);
        continue;
      }
      float m = 0.f, l = 0.f;
      if (static_max) {
        // ---- static-max softmax: p = 2^s', no row max, no rescale; 32-column chunks, the TMEM load of
        // chunk c+1 in flight while chunk c is exponentiated; at D = 64 every 4th exp2 on the FMA pipe
        // (Cfg::kPolyExp; MUFU: 16 ex2/clk/SM = 1024 clk per 128x128 tile).
        float rs0 = 0.f, rs1 = 0.f;
        for (int j = 0; j < sq.n_tiles; ++j, ++g) {
          wait(&s_full[t], g & 1);
          tc_fence_after();
          const int valid = sq.len - j * kTileRows;    // keys of this tile that exist
          uint32_t sa[32], sb[32];
          tmem_ld32(tS, sa);
          tmem_wait_ld();
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            uint32_t(&cur)[32] = (c & 1) ? sb : sa;
            uint32_t(&nxt)[32] = (c & 1) ? sa : sb;
            if (c < 3) tmem_ld32(tS + (c + 1) * 32, nxt);
            uint32_t pk[16];
            if (valid >= kTileRows) {
#pragma unroll
              for (int i = 0; i < 32; i += 2) {
                float p0, p1;
                if (Cfg::kPolyExp && (i & 2)) ex2_poly3_x2(__uint_as_float(cur[i]), __uint_as_float(cur[i + 1]), p0, p1);
                else { p0 = ex2_approx(__uint_as_float(cur[i])); p1 = ex2_approx(__uint_as_float(cur[i + 1])); }
                rs0 += p0; rs1 += p1;
                pk[i >> 1] = pack_bf16x2(p0, p1);
              }
            } else {
#pragma unroll
              for (int i = 0; i < 32; i += 2) {
                const float p0 = (c * 32 + i < valid) ? ex2_approx(__uint_as_float(cur[i])) : 0.f;
                const float p1 = (c * 32 + i + 1 < valid) ? ex2_approx(__uint_as_float(cur[i + 1])) : 0.f;
                rs0 += p0; rs1 += p1;
                pk[i >> 1] = pack_bf16x2(p0, p1);
              }
            }
            tmem_st16(tS + c * 16, pk);      // P (bf16 pairs) over S columns that have already been read
            if (kSplitP > 1 && c < 3 && ((c + 1) * kSplitP) % 4 == 0) {      // a piece of P is complete: hand it to the MMA warp now
              tmem_wait_st();
              tc_fence_before();
              arrive_mma(&pa_full[t * (kSplitP - 1) + (c + 1) * kSplitP / 4 - 1]);
            }
            if (c < 3) tmem_wait_ld();
          }
          tmem_wait_st();
          tc_fence_before();
          arrive_mma(&p_full[t]);
        }
        l = rs0 + rs1;
      } else {
        m = -INFINITY;
        for (int j = 0; j < sq.n_tiles; ++j, ++g) {
          wait(&s_full[t], g & 1);
          tc_fence_after();
          uint32_t su[128];
#pragma unroll
          for (int c = 0; c < 4; ++c) tmem_ld32(tS + c * 32, *reinterpret_cast<uint32_t(*)[32]>(&su[c * 32]));
          tmem_wait_ld();
          const int valid = sq.len - j * kTileRows;    // keys of this tile that exist
          if (valid < kTileRows) {
#pragma unroll
            for (int c = 0; c < 128; ++c) if (c >= valid) su[c] = 0xff800000u;   // -inf
          }
          float mx0 = __uint_as_float(su[0]), mx1 = __uint_as_float(su[1]);
#pragma unroll
          for (int c = 2; c < 128; c += 2) {
            mx0 = fmaxf(mx0, __uint_as_float(su[c]));
            mx1 = fmaxf(mx1, __uint_as_float(su[c + 1]));
          }
          const float m_new = fmaxf(m, fmaxf(mx0, mx1));
          float alpha = 1.0f;
          // lazy rescale: keep the stale max unless it is more than 8 (log2 units) too small
          const bool bump = (m_new - m) > 8.0f;     // true on the first tile (m = -inf)
          if (bump) { alpha = ex2_approx(m - m_new); m = m_new; }
          float rs0 = 0.f, rs1 = 0.f;
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) {
            uint32_t pk[16];
#pragma unroll
            for (int c = 0; c < 32; c += 2) {
              const float p0 = ex2_approx(__uint_as_float(su[q4 * 32 + c]) - m);
              const float p1 = ex2_approx(__uint_as_float(su[q4 * 32 + c + 1]) - m);
              rs0 += p0; rs1 += p1;
              pk[c >> 1] = pack_bf16x2(p0, p1);
            }
            tmem_st16(tS + q4 * 16, pk);
          }
          l = l * alpha + (rs0 + rs1);
          if (j > 0 && __any_sync(0xffffffffu, bump)) {
            // O += P V of tile g-1 must have completed before O is rescaled
            wait(&pv_done[t], (g - 1) & 1);
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
          for (int i = 0; i < kSplitP - 1; ++i) arrive_mma(&pa_full[t * (kSplitP - 1) + i]);   // (O may have been rescaled above: no early hand-off on this path)
          arrive_mma(&p_full[t]);
        }
      }
      // ---- epilogue: O / l -> bf16, LSE (natural log, reading R9)
      wait(&pv_done[t], (g - 1) & 1);
      tc_fence_after();
      const int t_item = (kCl ? 2 * static_cast<int>(rank) : 0) + t;     // this tile's place in the item (cluster forms: phantoms beyond wi.pad)
      const int n = (wi.tile + t_item) * kTileRows + row;     // token inside the sequence
      const int tok_g = sq.tok_start + n;
      const bool valid_row = t_item < wi.pad && n < sq.len && tok_g >= pd.cp_lo && tok_g < pd.cp_hi;   // CP: only this rank's query rows
      const float inv_l = 1.0f / l;
      __nv_bfloat16* orow = valid_row ? raw_row<__nv_bfloat16>(pd.sh, fp.o, sq.tok_start + n, wi.head, D) : nullptr;
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
      arrive_mma(&o_free[t]);
    }
  }
  tc_fence_before();
  if constexpr (kCl) cluster_sync_all(); else __syncthreads();   // (cluster: no remote arrival or multicast may target a CTA that has exited)
  if (pd.cta_trace && threadIdx.x == 0) pd.cta_trace[(0 * kTraceMaxCtas + blockIdx.x) * 2 + 1] = globaltimer_ns();
  if (warp == 9) {
    if constexpr (kPair) tmem_dealloc2(tbase, 512); else tmem_dealloc(tbase, 512);
  }
}

template <int D, bool kFusedQ = false>
__global__ void __launch_bounds__(320, 1) fwd_kernel(ProblemDesc pd, FwdParams fp, const __grid_constant__ RawMaps vmaps,
                                                      const __grid_constant__ RawMaps qmaps) {
  fwd_body<D, kFwdSingle, kFusedQ>(pd, fp, vmaps, qmaps);
}
// CTA-pair form: grid = 2 x (number of pairs), static cluster of 2 (the two SMs of a TPC)
template <int D>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(320, 1) fwd_pair_kernel(ProblemDesc pd, FwdParams fp,
                                                                                         const __grid_constant__ RawMaps vmaps) {
  fwd_body<D, kFwdPair>(pd, fp, vmaps, vmaps);      // (the pair form reads V images; the maps are unused)
}
// Multicast form: grid = 2 x (number of clusters), static cluster of 2
template <int D>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(320, 1) fwd_mc_kernel(ProblemDesc pd, FwdParams fp,
                                                                                       const __grid_constant__ RawMaps vmaps) {
  fwd_body<D, kFwdMcast>(pd, fp, vmaps, vmaps);
}

}  // namespace arachne
