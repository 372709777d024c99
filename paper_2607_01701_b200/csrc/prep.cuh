// Elementwise (HBM / issue-bound) kernels around the tensor-core kernels:
//   prep_kernel : §8 a1 + a5.  raw Q,K -> RMSNorm -> 3D RoPE -> fp16 operand tile images; backward: D_i = rowsum(dO*O),
//                 LSE*log2e (padded), per-group maxima for the dS / fixed-point scales; V, dO -> tile images (zero-padded
//                 tails) ONLY in the copy variant (sharded plans, ARACHNE_FLAG_IMAGE_COPIES) — otherwise the main kernels read
//                 them from the raw tensors by tensor-map TMA (rawtile.cuh).
//   post_kernel : §8 a8.  dq~, dk~ (fp32, or int32 fixed point) -> un-RoPE -> RMSNorm backward -> bf16 dQ, dK (+ dgamma
//                 partials, R22).
// Thread mapping: a lane owns 8 contiguous elements (one 16-byte bf16 load / store, one swizzle chunk of a tile
// image), so a (token, head) row takes LPR = D/8 lanes and a warp works on RPW = 32/LPR rows at once (2 at D = 128,
// 4 at D = 64).  Both elements of every RoPE pair (2p, 2p+1) sit in the same lane; the only cross-lane work is the
// sum over the LPR lanes of a row.  Token positions come from the plan's per-token table (TokInfo) — no integer
// divisions and no search over cu_seqlens on the device.  prep_kernel: one block per (tile, head); post_kernel: token-major
// with an inner loop over heads.  Both are bound by instruction issue as much as by HBM (profiles/r1_notes.md §7,
// profiles/r2_prologue.md).
#pragma once
#include "common.cuh"
#include "normrope.cuh"
#include "sm100.cuh"

namespace arachne {

struct PrepParams {
  ShardedPtr q, k, v;          // raw bf16 [N, H_total, D], possibly sharded by token range (common.cuh)
  ShardedPtr d_o, o;           // backward only
  const float* lse;            // nullable (forward)
  const float* gamma_q;        // nullable => ones
  const float* gamma_k;
  uint8_t* qt;                 // [H][n_tiles][128*D*2]
  uint8_t* kt;
  uint8_t* vt;                 // nullable: no V image (the main kernels read V by tensor-map TMA, rawtile.cuh)
  uint8_t* dot;                // nullable: forward, or no dO image (same)
  float* lse2_t;               // [H][n_tiles][128]  lse * log2(e); +inf on pad rows
  float* delta_t;              // [H][n_tiles][128]  rowsum(dO*O);  0 on pad rows
  float* gq_zero;              // nullable: blocked dq~ accumulator [H][n_tiles][128*D] to clear (fused backward)
  float* rowqs_t;              // nullable (deterministic backward): [H][n_tiles][128] out: |dO_i| of every query row, 0 on pad rows;
                               // bwd_scale_kernel turns it in place into the row's fixed-point scale (bwd_fused.cuh)
  float q_prescale;            // Q^ is multiplied by softmax_scale*log2(e) before it is rounded to fp16, so that S leaves the
                               // tensor core already in the exp2 domain — in the forward AND in the backward's recompute, which
                               // therefore sees bit-identical operands (P = exp2(S - LSE) consistent with the stored LSE)
  int skip_q;                  // forward, ARACHNE_FLAG_FWD_FUSED_Q: no Q^ image (fwd_kernel normalises its own query tiles)
  unsigned* stats;             // nullable (forward): [0] = max_i |q~'_i|^2, [1] = max_j |k~_j|^2 as float bits (atomicMax);
                               // the forward kernel derives its logit bound from them (static-max softmax)
};

// kCopy: also write V (and, backward, dO) tile images — the path of token-range-sharded plans and of ARACHNE_FLAG_IMAGE_COPIES;
// otherwise the main kernels read those tiles from the raw tensors by tensor-map TMA (rawtile.cuh) and pp.vt / pp.dot are null.
template <int D, bool kBwd, bool kCopy>
__global__ void __launch_bounds__(256, 4) prep_kernel(ProblemDesc pd, PrepParams pp) {
  constexpr int LPR = D / 8, RPW = 32 / LPR;
  constexpr int TILE_BYTES = kTileRows * D * 2;
  const int gtile = blockIdx.x, h = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int sub = lane / LPR, d0 = (lane % LPR) * 8;
  float qn = 0.f, kn = 0.f;      // largest |q~|^2, |k~|^2 seen by this lane's rows (no_norm only)
  float gn = 0.f, vn = 0.f;      // backward: largest |dO_i|^2, |V_j|^2 seen by this lane's rows (bound on dS, bwd_scale_kernel)
  const SeqInfo sq = pd.seqs[pd.tile_seq[gtile]];
  const int t = gtile - sq.tile_base;
  const size_t img_off = (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * TILE_BYTES;
  const size_t row_off = (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * kTileRows;
  // Context parallelism: K^ / V images are needed for every tile of a sequence this rank touches, the QUERY-side data
  // (Q^ image, dO image, lse2, delta, the dq~ accumulator) only for the tiles that hold some of the rank's own rows.
  const bool touched = sq.qt_n > 0;                              // a sequence without rows of this rank: nothing to prepare
  const bool q_side = t >= sq.qt_lo && t < sq.qt_lo + sq.qt_n && !pp.skip_q;   // always true without CP / fused Q
  if (pp.gq_zero && q_side) {
    float4* z = reinterpret_cast<float4*>(pp.gq_zero + (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * (kTileRows * D));
    for (int i = threadIdx.x; i < kTileRows * D / 4; i += 256) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  float gq[8], gk[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    gq[i] = pp.gamma_q ? __ldg(&pp.gamma_q[d0 + i]) : 1.0f;
    gk[i] = pp.gamma_k ? __ldg(&pp.gamma_k[d0 + i]) : 1.0f;
  }
  const uint4 zero4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll 1
  for (int r = warp * RPW + sub; touched && r < kTileRows; r += 8 * RPW) {
    const int n = t * kTileRows + r;            // token index inside the sequence
    const bool valid = n < sq.len;
    const int tok = sq.tok_start + (valid ? n : 0);
    const TokInfo ti = pd.tok_info[tok];
    const bool rotate = !pd.no_rope && !(ti.t_flag >> 31);   // R21: trailing text tokens are normed, not rotated
    int shard = 0;
    const long long dense = static_cast<long long>(pd.sh.H_total) * D;
    const size_t src = raw_off(pd.sh, dense, tok, h, D, shard) + d0;          // row in a contiguous tensor (dO, O)
    const long long trow = tok - pd.sh.start[shard];                            // Q, K, V may be token-strided (ProblemDesc::in_stride)
    uint4 uq = zero4, uk = zero4, uv = zero4, ug = zero4, uo = zero4;
    if (valid) {
      if (q_side) uq = *reinterpret_cast<const uint4*>(shard_base<const __nv_bfloat16>(pp.q, shard) + src + trow * (pd.in_stride[0] - dense));
      uk = *reinterpret_cast<const uint4*>(shard_base<const __nv_bfloat16>(pp.k, shard) + src + trow * (pd.in_stride[1] - dense));
      if (kBwd || kCopy) uv = *reinterpret_cast<const uint4*>(shard_base<const __nv_bfloat16>(pp.v, shard) + src + trow * (pd.in_stride[2] - dense));   // (bwd: |V|^2 bound)
      if (kBwd && q_side) {
        ug = *reinterpret_cast<const uint4*>(shard_base<const __nv_bfloat16>(pp.d_o, shard) + src);
        uo = *reinterpret_cast<const uint4*>(shard_base<const __nv_bfloat16>(pp.o, shard) + src);
      }
    }
    float2 cs[4];
    rope_cs4(pd.rope, d0, ti, rotate, cs);
    float xq[8], xk[8];
    unpack_bf16x8(uq, xq);
    unpack_bf16x8(uk, xk);
    const float qs = norm_rope8<D>(xq, gq, cs, pd.no_norm != 0, pd.eps, pp.q_prescale);
    const float ks = norm_rope8<D>(xk, gk, cs, pd.no_norm != 0, pd.eps, 1.0f);
    const uint32_t ioff = image_off(r, d0);
    if (q_side) *reinterpret_cast<uint4*>(pp.qt + img_off + ioff) = valid ? pack8(xq, FMT_F16) : zero4;   // (eps = 0: 0 * inf)
    *reinterpret_cast<uint4*>(pp.kt + img_off + ioff) = valid ? pack8(xk, FMT_F16) : zero4;
    if (kCopy) *reinterpret_cast<uint4*>(pp.vt + img_off + ioff) = uv;          // bf16 -> bf16 is exact
    // row norms are only needed when RMSNorm is off; with it on, |x^|^2 <= D * max(gamma)^2 (see below)
    if (pp.stats && pd.no_norm) { qn = fmaxf(qn, seg_sum<LPR>(qs)); kn = fmaxf(kn, seg_sum<LPR>(ks)); }
    if (kBwd && pd.no_norm) kn = fmaxf(kn, seg_sum<LPR>(ks));      // (with RMSNorm the bound D * max gamma_k^2 is used: bwd_scale_kernel)
    if (kBwd) {
      float vv[8], v2 = 0.f;
      unpack_bf16x8(uv, vv);
#pragma unroll
      for (int i = 0; i < 8; ++i) v2 += vv[i] * vv[i];
      vn = fmaxf(vn, seg_sum<LPR>(v2));
    }
    if (kBwd && q_side) {
      if (kCopy) *reinterpret_cast<uint4*>(pp.dot + img_off + ioff) = ug;
      float g[8], oo[8];
      unpack_bf16x8(ug, g);
      unpack_bf16x8(uo, oo);
      float dsum = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) dsum += g[i] * oo[i];
      dsum = seg_sum<LPR>(dsum);                                // D_i = sum_d dO*O   (§8 a5)
      float g2 = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) g2 += g[i] * g[i];
      g2 = seg_sum<LPR>(g2);
      gn = fmaxf(gn, g2);
      if (d0 == 0) {
        // context parallelism: query rows of other ranks behave like pad rows here (P = 0: no dK/dV contribution)
        const bool live = valid && tok >= pd.cp_lo && tok < pd.cp_hi;
        pp.delta_t[row_off + r] = live ? dsum : 0.f;
        if (pp.rowqs_t) pp.rowqs_t[row_off + r] = live ? sqrtf(g2) : 0.f;
        // pad rows get +inf so that P = exp2(s - inf) = 0 for them in the backward kernels
        pp.lse2_t[row_off + r] = live ? pp.lse[static_cast<size_t>(h) * pd.N + tok] * 1.4426950408889634f
                                       : __int_as_float(0x7f800000);
      }
    }
  }
  if (kBwd && touched) {
    // per (sequence, head) group: max_i |dO_i|^2 and max_j |V_j|^2 (non-negative floats order like their bit patterns;
    // NaN / inf sort last and make bwd_scale_kernel fall back to sk = 1)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      gn = fmaxf(gn, __shfl_xor_sync(0xffffffffu, gn, o));
      vn = fmaxf(vn, __shfl_xor_sync(0xffffffffu, vn, o));
    }
    if (lane == 0) {
      unsigned* gs = pd.grp_stats + (static_cast<size_t>(pd.tile_seq[gtile]) * pd.H + h) * 4;
      atomicMax(&gs[0], __float_as_uint(gn));
      atomicMax(&gs[1], __float_as_uint(vn));
      if (pd.no_norm) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) kn = fmaxf(kn, __shfl_xor_sync(0xffffffffu, kn, o));
        atomicMax(&gs[2], __float_as_uint(kn));
      }
    }
  }
  if (pp.stats) {
    // Bound on |q~'|^2 and |k~|^2 for the forward kernel's static-max softmax.  With RMSNorm,
    // |x^|^2 = sum_d gamma_d^2 x_d^2 / (mean(x^2) + eps) <= D * max_d gamma_d^2 (RoPE preserves the norm),
    // identical for every block, so one warp publishes it; without it, the largest row norm seen.
    // Non-negative floats order like their bit patterns (+inf sorts last -> online-softmax path).
    if (!pd.no_norm) {
      if (blockIdx.x == 0 && blockIdx.y == 0 && warp == 0) {
        float mq = 0.f, mk = 0.f;
        for (int d = lane; d < D; d += 32) {
          mq = fmaxf(mq, pp.gamma_q ? fabsf(pp.gamma_q[d]) : 1.0f);
          mk = fmaxf(mk, pp.gamma_k ? fabsf(pp.gamma_k[d]) : 1.0f);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          mq = fmaxf(mq, __shfl_xor_sync(0xffffffffu, mq, o));
          mk = fmaxf(mk, __shfl_xor_sync(0xffffffffu, mk, o));
        }
        if (lane == 0) {
          atomicMax(&pp.stats[0], __float_as_uint(mq * mq * D * pp.q_prescale * pp.q_prescale));
          atomicMax(&pp.stats[1], __float_as_uint(mk * mk * D));
        }
      }
    } else {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        qn = fmaxf(qn, __shfl_xor_sync(0xffffffffu, qn, o));
        kn = fmaxf(kn, __shfl_xor_sync(0xffffffffu, kn, o));
      }
      if (lane == 0) {
        atomicMax(&pp.stats[0], __float_as_uint(qn));
        atomicMax(&pp.stats[1], __float_as_uint(kn));
      }
    }
  }
}

// dS scaling for the fp16 backward GEMMs.  The backward recomputes S from the SAME fp16 Q^', K^ images as the
// forward, so dS must be fp16 too (tcgen05 kind::f16 takes one 16-bit format per instruction pair of operands); fp16 has 5
// exponent bits, so dS is multiplied by a power of two sk chosen per (sequence, head) group from a rigorous bound:
//   |dS_ij| = P_ij |dO_i.V_j - dO_i.O_i| <= 2 max_i|dO_i| max_j|V_j|      (P_ij <= 1; O_i is a convex combination of the V_j)
//   sk = 2^floor(log2(32768 / (2.02 max|dO| max|V|)))   =>   |dS sk| <= 32768 < 65504, never overflows;
// entries more than 2^-29 below the bound lose relative (not absolute) precision in fp16 subnormals — their absolute error,
// 2^-25/sk, stays ~2^16 times below bf16's at the bound.  The factor is folded into delta (this kernel) and the dP FFMA.
// Grid (n_tiles_total, H), 128 threads (one row each).
__global__ void __launch_bounds__(128) bwd_scale_kernel(ProblemDesc pd, float* delta_t, const float* gamma_k, int D, float* rowqs_t) {
  const int gtile = blockIdx.x, h = blockIdx.y;
  const int b = pd.tile_seq[gtile];
  const size_t g = static_cast<size_t>(b) * pd.H + h;
  const float gn = __uint_as_float(pd.grp_stats[g * 4]), vn = __uint_as_float(pd.grp_stats[g * 4 + 1]);
  const float bound = 2.02f * sqrtf(gn) * sqrtf(vn);
  float sk = 1.0f;
  if (bound > 0.f && bound < 3.0e38f) {      // (false for NaN)
    int e = static_cast<int>(floorf(log2f(32768.0f / bound)));
    e = max(-60, min(60, e));
    sk = exp2f(static_cast<float>(e));
  }
  const size_t row = (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * kTileRows + threadIdx.x;
  delta_t[row] *= sk;
  if (threadIdx.x == 0 && gtile == pd.seqs[b].tile_base) *reinterpret_cast<float2*>(pd.grp_sk + g * 4) = make_float2(sk, 1.0f / sk);
  if (rowqs_t) {
    // Fixed-point scale of the deterministic dq~ reduction (bwd_fused.cuh), one per QUERY ROW: every partial sum of
    // softmax_scale * dS_i. k~ over the keys, in any order, is bounded by softmax_scale * B_i,
    //   B_i = 2 |dO_i| max_j|V_j| * max_j |k~_j|,   |k~_j|^2 <= D * max_d gamma_k[d]^2 under RMSNorm (RoPE preserves the norm),
    // else the measured row maximum.  The scale follows the row's OWN |dO_i| (prep_kernel left it in rowqs_t), so a token with
    // an outlying upstream gradient takes resolution from nobody else: each row keeps ~30 bits below its own bound.
    __shared__ float s_gm[4];
    float kn = __uint_as_float(pd.grp_stats[g * 4 + 2]);
    if (!pd.no_norm) {
      float gm = 1.0f;
      if (gamma_k) {
        gm = threadIdx.x < D ? fabsf(gamma_k[threadIdx.x]) : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) gm = fmaxf(gm, __shfl_xor_sync(0xffffffffu, gm, o));
        if ((threadIdx.x & 31) == 0) s_gm[threadIdx.x >> 5] = gm;
        __syncthreads();
        gm = fmaxf(fmaxf(s_gm[0], s_gm[1]), fmaxf(s_gm[2], s_gm[3]));
      }
      kn = gm * gm * static_cast<float>(D);
    }
    const float bq = 1.01f * pd.softmax_scale * 2.02f * rowqs_t[row] * sqrtf(vn) * sqrtf(kn);
    float qs = 1.0f;                          // |dO_i| = 0 (pad rows too): every partial is exactly 0
    if (bq > 0.f && bq < 3.0e38f) {           // (false for NaN: the drain then marks the row, bwd_fused.cuh)
      int e = static_cast<int>(floorf(log2f(1073741824.0f / bq)));      // 2^30: headroom for the rounding of every partial
      e = max(-90, min(90, e));
      qs = exp2f(static_cast<float>(e));
    }
    rowqs_t[row] = qs;
  }
}

struct PostParams {
  const float* gq_t;            // dl/dq~ fp32 (already multiplied by softmax_scale): [N,H,D], or if gq_blocked the
                                // blocked/swizzled per-tile layout written by bwd_fused_kernel (gq_blk_off)
  int gq_blocked;
  int gq_fixed;                 // gq_t holds int32 fixed point (deterministic backward): value = int / rowqs_t[head][blocked row]
  const float* gk_t;
  ShardedPtr q, k;              // raw bf16, possibly sharded (common.cuh)
  const float* gamma_q;
  const float* gamma_k;
  ShardedPtr dq, dk;            // out bf16, same sharding
  int which;                    // 0: y = 0 -> dQ, y = 1 -> dK;  1: dQ only (grid.y = 1);  2: dK only (grid.y = 1)
  int tok_lo, tok_hi;           // only (token, head) rows with tok in [tok_lo, tok_hi) are processed (CP; else 0, N)
  float* dgamma_part;           // nullable: [2][gridDim.x][D] per-block partial sums of dl/dgamma_q, dl/dgamma_k (R22)
  const float* rowqs_t;         // gq_fixed: [H][n_tiles][128] fixed-point scale of every query row (a power of two; NaN = the row
                                // overflowed or saw a non-finite partial: its dQ is NaN, bwd_fused.cuh)
};

// dx = r*u - r^3 * x * (sum_d u_d x_d)/D,  u = gamma * R^T g~   (§8 a8; oracle: norm_rope_row_bwd)
// dl/dgamma_d += (R^T g~)_d * x_d * r                            (reading R22)
// Grid (nblk, 2): y = 0 -> dQ, y = 1 -> dK.  TOKEN-major: a warp takes RPW tokens per step (grid stride over the token groups)
// and walks ALL heads of them in an inner loop, so everything that depends on the token only — its TokInfo, the cos / sin of
// its RoPE pairs, its shard and row offsets, its place in the blocked dq~ layout — is set up once per token instead of once
// per (token, head) row, and consecutive iterations read consecutive 2*D-byte rows of the raw tensor (the kernel was
// instruction-issue-bound, ~390 instructions per row pair: profiles/r2_prologue.md).  A lane's dgamma partial stays in
// registers until the end; the per-block partials are then summed in block order by dgamma_reduce_kernel (fixed order:
// run-to-run bit-reproducible for a given plan, whichever backward produced g~).
// (4 blocks / SM and no unrolling of the head loop measured best: occupancy matters more than ILP here; 3 blocks / SM without
// the 40-byte spill is 20 % slower, profiles/r2_prologue.md)
template <int D>
__global__ void __launch_bounds__(256, 4) post_kernel(ProblemDesc pd, PostParams pp) {
  constexpr int LPR = D / 8, RPW = 32 / LPR;
  __shared__ float s_part[8 * RPW][D];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sub = lane / LPR, d0 = (lane % LPR) * 8;
  const bool is_k = pp.which == 2 || blockIdx.y == 1;
  const float* gt = is_k ? pp.gk_t : pp.gq_t;
  const ShardedPtr& xraw_s = is_k ? pp.k : pp.q;
  const float* gamma = is_k ? pp.gamma_k : pp.gamma_q;
  const ShardedPtr& out_s = is_k ? pp.dk : pp.dq;
  const bool blocked = !is_k && pp.gq_blocked;
  float gam[8], dgam[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { gam[i] = gamma ? __ldg(&gamma[d0 + i]) : 1.0f; dgam[i] = 0.f; }
  const long long dense = static_cast<long long>(pd.sh.H_total) * D;
  const size_t blk_head_stride = static_cast<size_t>(pd.n_tiles_total) * (kTileRows * D);     // floats between heads, blocked dq~
  const int stride = gridDim.x * 8 * RPW;
  for (int tok0 = pp.tok_lo + (blockIdx.x * 8 + warp) * RPW; tok0 < pp.tok_hi; tok0 += stride) {   // warp-uniform trip count
    const bool live = tok0 + sub < pp.tok_hi;                  // ragged end: the lane keeps shuffling, stores nothing
    const int tok = live ? tok0 + sub : pp.tok_hi - 1;
    // ---- per token
    const TokInfo ti = pd.tok_info[tok];
    const bool rotate = !pd.no_rope && !(ti.t_flag >> 31);     // R21: text tokens were not rotated
    float2 cs[4];
    rope_cs4(pd.rope, d0, ti, rotate, cs);
    int shard;
    const size_t roff0 = raw_off(pd.sh, dense, tok, 0, D, shard) + d0;                                        // output row of head 0 (contiguous)
    const size_t xoff0 = roff0 + static_cast<long long>(tok - pd.sh.start[shard]) * (pd.in_stride[is_k ? 1 : 0] - dense);   // raw Q / K row (may be token-strided)
    const __nv_bfloat16* xbase = shard_base<const __nv_bfloat16>(xraw_s, shard) + xoff0;
    __nv_bfloat16* obase = shard_base<__nv_bfloat16>(out_s, shard) + roff0;
    const float* g0p; const float* g1p; size_t gstep;
    if (blocked) {
      // blocked layout [H][tile][D/32][128 rows][32], 16-byte pieces XOR-swizzled with (row & 7) (bwd_fused.cuh)
      const int qr = ti.blkrow & (kTileRows - 1), j = (d0 & 31) >> 2;
      const float* base = gt + static_cast<size_t>(ti.blkrow >> 7) * (kTileRows * D) + static_cast<size_t>(d0 >> 5) * (kTileRows * 32) + qr * 32;
      g0p = base + ((j ^ (qr & 7)) << 2); g1p = base + (((j + 1) ^ (qr & 7)) << 2); gstep = blk_head_stride;
    } else {
      g0p = gt + static_cast<size_t>(tok) * pd.H * D + d0; g1p = g0p + 4; gstep = D;      // local fp32 workspace [N, H, D]
    }
    const float* iqp = pp.gq_fixed && blocked ? pp.rowqs_t + ti.blkrow : nullptr;
    const size_t iq_head_stride = static_cast<size_t>(pd.n_tiles_total) * kTileRows;
    // ---- per (token, head) row
#pragma unroll 1
    for (int h = 0; h < pd.H; ++h) {
      const uint4 ux = *reinterpret_cast<const uint4*>(xbase + static_cast<size_t>(h) * D);
      float4 f0 = *reinterpret_cast<const float4*>(g0p + h * gstep);
      float4 f1 = *reinterpret_cast<const float4*>(g1p + h * gstep);
      if (iqp) {      // int32 fixed point (deterministic backward): value = int / qs of this (token, head) row
        const float qsv = iqp[h * iq_head_stride];
        // qs = 2^e, |e| <= 90: its reciprocal is the mirrored exponent field (exact); a NaN mark stays NaN
        const float iq = qsv == qsv ? __uint_as_float(0x7f000000u - __float_as_uint(qsv)) : qsv;
        f0 = make_float4(__float_as_int(f0.x) * iq, __float_as_int(f0.y) * iq, __float_as_int(f0.z) * iq, __float_as_int(f0.w) * iq);
        f1 = make_float4(__float_as_int(f1.x) * iq, __float_as_int(f1.y) * iq, __float_as_int(f1.z) * iq, __float_as_int(f1.w) * iq);
      }
      float g[8] = {f0.x, f0.y, f0.z, f0.w, f1.x, f1.y, f1.z, f1.w};
      float x[8];
      unpack_bf16x8(ux, x);
#pragma unroll
      for (int i = 0; i < 8; i += 2) {
        const float2 c = cs[i >> 1];
        const float ga = g[i], gb = g[i + 1];
        g[i] = ga * c.x + gb * c.y;          // rotate by -phi
        g[i + 1] = -ga * c.y + gb * c.x;
      }
      float y[8];
      if (!pd.no_norm) {
        float ss = 0.f, uxs = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          ss += x[i] * x[i];
          uxs += gam[i] * g[i] * x[i];
        }
        ss = seg_sum<LPR>(ss);
        uxs = seg_sum<LPR>(uxs);
        const float rinv = rsqrtf(ss * (1.0f / D) + pd.eps);
        const float c = rinv * rinv * rinv * uxs * (1.0f / D);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          y[i] = rinv * gam[i] * g[i] - c * x[i];
          if (live) dgam[i] += g[i] * x[i] * rinv;
        }
      } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) y[i] = g[i];      // gamma unused: dgamma = 0
      }
      if (live) *reinterpret_cast<uint4*>(obase + static_cast<size_t>(h) * D) = pack8(y, FMT_BF16);
    }
  }
  if (pp.dgamma_part) {
#pragma unroll
    for (int i = 0; i < 8; ++i) s_part[warp * RPW + sub][d0 + i] = dgam[i];
    __syncthreads();
    if (threadIdx.x < D) {
      float a = 0.f;
#pragma unroll
      for (int w = 0; w < 8 * RPW; ++w) a += s_part[w][threadIdx.x];
      pp.dgamma_part[(static_cast<size_t>(is_k ? 1 : 0) * gridDim.x + blockIdx.x) * D + threadIdx.x] = a;
    }
  }
}

// dgamma[d] = sum over the post_kernel blocks, in block order.  Grid 2 (0: gamma_q, 1: gamma_k), 256 threads:
// thread (s, d) with s = tid / D sums the blocks b == s (mod 256/D); the 256/D slices are then added in order.
template <int D>
__global__ void __launch_bounds__(256) dgamma_reduce_kernel(const float* part, int nblk, float* dgamma_q, float* dgamma_k) {
  constexpr int S = 256 / D;
  __shared__ float s[S][D];
  const int d = threadIdx.x % D, sl = threadIdx.x / D;
  const float* p = part + static_cast<size_t>(blockIdx.x) * nblk * D;
  float a = 0.f;
  for (int b = sl; b < nblk; b += S) a += p[static_cast<size_t>(b) * D + d];
  s[sl][d] = a;
  __syncthreads();
  float* out = blockIdx.x == 0 ? dgamma_q : dgamma_k;
  if (sl == 0 && out) {
    float t = 0.f;
#pragma unroll
    for (int i = 0; i < S; ++i) t += s[i][d];
    out[d] = t;
  }
}


// Context parallelism, phase 2 ("CP ... sequence partition"): every rank has written
// PARTIAL dk~ and dV (fp32 [N,H,D], from its own query rows) for all keys of the sequences it touches.  The owner of a
// key token adds the partials of the contributing ranks IN RANK ORDER (fixed order: bit-reproducible) — reading them
// straight out of the peers' buffers (the reduce-scatter is these loads) — and emits dV (bf16) and the summed dk~ for
// post_kernel.  Rank r contributes to a token iff its query range intersects the token's sequence.
struct CpReduceParams {
  ShardedPtr gk_part, gv_part;   // [n_shards] fp32 [N,H,D] partial buffers, one per rank (local or peer memory)
  float* gk_sum;                 // out: fp32 [N,H,D], rows [tok_lo, tok_hi) only
  ShardedPtr dv;                 // out: bf16, token-range sharded like every raw tensor
  int tok_lo, tok_hi;
};

template <int D>
__global__ void __launch_bounds__(256) cp_reduce_kernel(ProblemDesc pd, CpReduceParams cp) {
  constexpr int VPR = D / 4;                                       // float4 pieces per (token, head) row
  const long long n_vec = static_cast<long long>(cp.tok_hi - cp.tok_lo) * pd.H * VPR;
  for (long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; i < n_vec;
       i += static_cast<long long>(gridDim.x) * blockDim.x) {
    const int piece = static_cast<int>(i % VPR);
    const long long rh = i / VPR;
    const int tok = cp.tok_lo + static_cast<int>(rh / pd.H), h = static_cast<int>(rh % pd.H);
    const SeqInfo sq = pd.seqs[pd.tok_info[tok].seq];
    const size_t off = (static_cast<size_t>(tok) * pd.H + h) * D + piece * 4;
    float4 sk = make_float4(0.f, 0.f, 0.f, 0.f), sv = sk;
#pragma unroll
    for (int r = 0; r < kMaxShards; ++r) {
      if (r < pd.sh.n_shards && pd.sh.start[r + 1] > pd.sh.start[r] && pd.sh.start[r] < sq.tok_start + sq.len &&
          pd.sh.start[r + 1] > sq.tok_start) {
        const float4 a = *reinterpret_cast<const float4*>(shard_base<const float>(cp.gk_part, r) + off);
        const float4 b = *reinterpret_cast<const float4*>(shard_base<const float>(cp.gv_part, r) + off);
        sk.x += a.x; sk.y += a.y; sk.z += a.z; sk.w += a.w;
        sv.x += b.x; sv.y += b.y; sv.z += b.z; sv.w += b.w;
      }
    }
    *reinterpret_cast<float4*>(cp.gk_sum + off) = sk;
    uint2 u; u.x = pack_bf16x2(sv.x, sv.y); u.y = pack_bf16x2(sv.z, sv.w);
    *reinterpret_cast<uint2*>(raw_row<__nv_bfloat16>(pd.sh, cp.dv, tok, h, D) + piece * 4) = u;
  }
}

}  // namespace arachne
