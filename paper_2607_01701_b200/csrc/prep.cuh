// Elementwise (HBM-bound) kernels around the tensor-core kernels:
//   prep_kernel : §8 a1 + a5.  raw Q,K -> RMSNorm -> 3D RoPE -> 16-bit operand tile images;
//                 V, dO -> tile images (zero-padded tails); D_i = rowsum(dO*O); LSE*log2e padded.
//   post_kernel : §8 a8.  dq~, dk~ (fp32) -> un-RoPE -> RMSNorm backward -> bf16 dQ, dK.
// One warp owns one (token, head) row; lane l owns the D/32 contiguous elements [l*D/32, ...),
// so both elements of every RoPE pair (2p, 2p+1) sit in the same lane and the only cross-lane
// work is the sum of squares.  All loads/stores are whole 128/256-byte row segments.
#pragma once
#include "common.cuh"
#include "sm100.cuh"

namespace arachne {

struct PrepParams {
  ShardedPtr q, k, v;          // raw bf16 [N, H_total, D], possibly sharded by token range (common.cuh)
  ShardedPtr d_o, o;           // backward only
  int backward;                // 0 forward, 1 backward (d_o, o, lse valid)
  const float* lse;            // nullable (forward)
  const float* gamma_q;        // nullable => ones
  const float* gamma_k;
  uint8_t* qt;                 // [H][n_tiles][128*D*2]
  uint8_t* kt;
  uint8_t* vt;
  uint8_t* dot;                // nullable
  float* lse2_t;               // [H][n_tiles][128]  lse * log2(e); +inf on pad rows
  float* delta_t;              // [H][n_tiles][128]  rowsum(dO*O);  0 on pad rows
  float* gq_zero;              // nullable: blocked dq~ accumulator [H][n_tiles][128*D] to clear (fused backward)
  int out_fmt;                 // FMT_F16 (forward: LSE accuracy) or FMT_BF16 (backward)
  float q_prescale;            // Q^ is multiplied by this before rounding (forward: softmax_scale*log2(e), so that
                               // S comes out of the tensor core already in the exp2 domain; backward: 1)
  unsigned* stats;             // nullable: [0] = max_i |q~_i|^2, [1] = max_j |k~_j|^2 as float bits (atomicMax);
                               // the forward kernel derives its logit bound from them (static-max softmax)
};

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

template <int EPL>
__device__ __forceinline__ void load_bf16_row(const __nv_bfloat16* p, float (&x)[EPL]) {
  if constexpr (EPL == 4) {
    const uint2 u = *reinterpret_cast<const uint2*>(p);
    x[0] = __uint_as_float(u.x << 16); x[1] = __uint_as_float(u.x & 0xffff0000u);
    x[2] = __uint_as_float(u.y << 16); x[3] = __uint_as_float(u.y & 0xffff0000u);
  } else {
    const uint32_t u = *reinterpret_cast<const uint32_t*>(p);
    x[0] = __uint_as_float(u << 16); x[1] = __uint_as_float(u & 0xffff0000u);
  }
}

// (cos, sin) of the RoPE pair `pp` (0..D/2-1) at grid position pos[]
__device__ __forceinline__ float2 rope_cs(const RopeDesc& rp, int pp, const int (&pos)[3]) {
  int a = 0, p = pp;
  if (p >= rp.half[0]) { p -= rp.half[0]; a = 1; if (p >= rp.half[1]) { p -= rp.half[1]; a = 2; } }
  return __ldg(&rp.tab[rp.off[a] + pos[a] * rp.half[a] + p]);
}

// byte offset of element d of row r inside a [128][D] tile image
__device__ __forceinline__ uint32_t image_off(int r, int d) {
  return static_cast<uint32_t>(d >> 6) * (kTileRows * 128) + swz_off(r, (d & 63) >> 3) + (d & 7) * 2;
}

template <int EPL>
__device__ __forceinline__ void store_image(uint8_t* img, int r, int d0, const float (&y)[EPL], int fmt) {
  uint8_t* dst = img + image_off(r, d0);
  if constexpr (EPL == 4) {
    uint2 u;
    if (fmt == FMT_F16) { u.x = pack_f16x2(y[0], y[1]); u.y = pack_f16x2(y[2], y[3]); }
    else                { u.x = pack_bf16x2(y[0], y[1]); u.y = pack_bf16x2(y[2], y[3]); }
    *reinterpret_cast<uint2*>(dst) = u;
  } else {
    *reinterpret_cast<uint32_t*>(dst) = fmt == FMT_F16 ? pack_f16x2(y[0], y[1]) : pack_bf16x2(y[0], y[1]);
  }
}

// x~ = RoPE(gamma * x * rsqrt(mean(x^2) + eps))  (readings R1-R5), one row per warp
// returns the lane's partial sum of squares of the stored row (0 for pad rows)
template <int D>
__device__ __forceinline__ float norm_rope_store(const ProblemDesc& pd, const __nv_bfloat16* src, const float* gamma,
                                                 uint8_t* img, int r, bool valid, bool rotate, const int (&pos)[3], int lane,
                                                 int fmt, float prescale) {
  constexpr int EPL = D / 32;
  const int d0 = lane * EPL;
  float x[EPL];
  float nrm = 0.f;
  if (valid) {
    load_bf16_row<EPL>(src + d0, x);
    if (!pd.no_norm) {
      float ss = 0.f;
#pragma unroll
      for (int i = 0; i < EPL; ++i) ss += x[i] * x[i];
      ss = warp_sum(ss);
      const float rinv = rsqrtf(ss * (1.0f / D) + pd.eps);
#pragma unroll
      for (int i = 0; i < EPL; ++i) x[i] *= rinv * (gamma ? __ldg(&gamma[d0 + i]) : 1.0f);
    }
    if (rotate) {
#pragma unroll
      for (int i = 0; i < EPL; i += 2) {
        const float2 cs = rope_cs(pd.rope, (d0 + i) >> 1, pos);
        const float x0 = x[i], x1 = x[i + 1];
        x[i] = x0 * cs.x - x1 * cs.y;
        x[i + 1] = x0 * cs.y + x1 * cs.x;
      }
    }
#pragma unroll
    for (int i = 0; i < EPL; ++i) { x[i] *= prescale; nrm += x[i] * x[i]; }
  } else {
#pragma unroll
    for (int i = 0; i < EPL; ++i) x[i] = 0.f;   // zero-padded tail rows (never NaN: 0 * P stays 0)
  }
  store_image<EPL>(img, r, d0, x, fmt);
  return nrm;
}

template <int D>
__global__ void __launch_bounds__(256) prep_kernel(ProblemDesc pd, PrepParams pp) {
  constexpr int EPL = D / 32;
  constexpr int TILE_BYTES = kTileRows * D * 2;
  const int gtile = blockIdx.x, h = blockIdx.y;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float qn = 0.f, kn = 0.f;      // this warp's largest |q~|^2, |k~|^2 (lane-partial sums until the end)
  const SeqInfo sq = pd.seqs[pd.tile_seq[gtile]];
  const int t = gtile - sq.tile_base;
  const size_t img_off = (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * TILE_BYTES;
  const size_t row_off = (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * kTileRows;
  const int d0 = lane * EPL;
  if (pp.gq_zero) {
    float4* z = reinterpret_cast<float4*>(pp.gq_zero + (static_cast<size_t>(h) * pd.n_tiles_total + gtile) * (kTileRows * D));
    for (int i = threadIdx.x; i < kTileRows * D / 4; i += 256) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  for (int r = warp; r < kTileRows; r += 8) {
    const int n = t * kTileRows + r;            // token index inside the sequence
    const bool valid = n < sq.len;
    const bool rotate = !pd.no_rope && n < sq.n_video;   // R21: trailing text tokens are normed, not rotated
    int pos[3];
    const int hw = sq.Hg * sq.Wg;
    pos[0] = n / hw; pos[1] = (n / sq.Wg) % sq.Hg; pos[2] = n % sq.Wg;   // only read when rotate
    int shard = 0;
    const size_t src = valid ? raw_off(pd.sh, sq.tok_start + n, h, D, shard) : 0;
    const __nv_bfloat16* qsrc = shard_base<const __nv_bfloat16>(pp.q, shard) + src;
    const __nv_bfloat16* ksrc = shard_base<const __nv_bfloat16>(pp.k, shard) + src;
    const float qs = norm_rope_store<D>(pd, qsrc, pp.gamma_q, pp.qt + img_off, r, valid, rotate, pos, lane, pp.out_fmt, pp.q_prescale);
    const float ks = norm_rope_store<D>(pd, ksrc, pp.gamma_k, pp.kt + img_off, r, valid, rotate, pos, lane, pp.out_fmt, 1.0f);
    // row norms are only summed when RMSNorm is off; with it on, |x^|^2 <= D * max(gamma)^2 (see below)
    if (pp.stats && pd.no_norm) { qn = fmaxf(qn, warp_sum(qs)); kn = fmaxf(kn, warp_sum(ks)); }
    float x[EPL];
    if (valid) load_bf16_row<EPL>(shard_base<const __nv_bfloat16>(pp.v, shard) + src + d0, x);
    else {
#pragma unroll
      for (int i = 0; i < EPL; ++i) x[i] = 0.f;
    }
    store_image<EPL>(pp.vt + img_off, r, d0, x, FMT_BF16);     // bf16 -> bf16 is exact
    if (pp.backward) {
      float g[EPL], oo[EPL];
      float dsum = 0.f;
      if (valid) {
        load_bf16_row<EPL>(shard_base<const __nv_bfloat16>(pp.d_o, shard) + src + d0, g);
        load_bf16_row<EPL>(shard_base<const __nv_bfloat16>(pp.o, shard) + src + d0, oo);
#pragma unroll
        for (int i = 0; i < EPL; ++i) dsum += g[i] * oo[i];
      } else {
#pragma unroll
        for (int i = 0; i < EPL; ++i) g[i] = 0.f;
      }
      store_image<EPL>(pp.dot + img_off, r, d0, g, FMT_BF16);
      dsum = warp_sum(dsum);                                    // D_i = sum_d dO*O   (§8 a5)
      if (lane == 0) {
        pp.delta_t[row_off + r] = valid ? dsum : 0.f;
        // pad rows get +inf so that P = exp2(s - inf) = 0 for them in the backward kernels
        pp.lse2_t[row_off + r] = valid ? pp.lse[static_cast<size_t>(h) * pd.N + sq.tok_start + n] * 1.4426950408889634f
                                       : __int_as_float(0x7f800000);
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
        float gq = 0.f, gk = 0.f;
        for (int d = lane; d < D; d += 32) {
          gq = fmaxf(gq, pp.gamma_q ? fabsf(pp.gamma_q[d]) : 1.0f);
          gk = fmaxf(gk, pp.gamma_k ? fabsf(pp.gamma_k[d]) : 1.0f);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          gq = fmaxf(gq, __shfl_xor_sync(0xffffffffu, gq, o));
          gk = fmaxf(gk, __shfl_xor_sync(0xffffffffu, gk, o));
        }
        if (lane == 0) {
          atomicMax(&pp.stats[0], __float_as_uint(gq * gq * D * pp.q_prescale * pp.q_prescale));
          atomicMax(&pp.stats[1], __float_as_uint(gk * gk * D));
        }
      }
    } else if (lane == 0) {
      atomicMax(&pp.stats[0], __float_as_uint(qn));
      atomicMax(&pp.stats[1], __float_as_uint(kn));
    }
  }
}

struct PostParams {
  const float* gq_t;            // dl/dq~ fp32 (already multiplied by softmax_scale): [N,H,D], or if gq_blocked the
                                // blocked/swizzled per-tile layout written by bwd_fused_kernel (gq_blk_off)
  int gq_blocked;
  const float* gk_t;
  ShardedPtr q, k;              // raw bf16, possibly sharded (common.cuh)
  const float* gamma_q;
  const float* gamma_k;
  ShardedPtr dq, dk;            // out bf16, same sharding
  float* dgamma_part;           // nullable: [2][gridDim.x][D] per-block partial sums of dl/dgamma_q, dl/dgamma_k (R22)
};

// dx = r*u - r^3 * x * (sum_d u_d x_d)/D,  u = gamma * R^T g~   (§8 a8; oracle: norm_rope_row_bwd)
// dl/dgamma_d += (R^T g~)_d * x_d * r                            (reading R22)
// Grid (nblk, 2): y = 0 -> dQ, y = 1 -> dK.  Warps walk the (token, head) rows with a grid stride, so a
// warp's dgamma partial stays in registers (lane l owns elements [l*D/32, ...)) until the end; the
// per-block partials are then summed in block order by dgamma_reduce_kernel (fixed order: run-to-run
// bit-reproducible for a given plan, whichever backward produced g~).
template <int D>
__global__ void __launch_bounds__(256) post_kernel(ProblemDesc pd, PostParams pp) {
  constexpr int EPL = D / 32;
  __shared__ float s_part[8][D];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool is_k = blockIdx.y == 1;
  const float* gt = is_k ? pp.gk_t : pp.gq_t;
  const ShardedPtr& xraw_s = is_k ? pp.k : pp.q;
  const float* gamma = is_k ? pp.gamma_k : pp.gamma_q;
  const ShardedPtr& out_s = is_k ? pp.dk : pp.dq;
  const int d0 = lane * EPL;
  float gam[EPL], dgam[EPL];
#pragma unroll
  for (int i = 0; i < EPL; ++i) { gam[i] = gamma ? __ldg(&gamma[d0 + i]) : 1.0f; dgam[i] = 0.f; }
  const long long n_rows = static_cast<long long>(pd.N) * pd.H;
  const long long stride = static_cast<long long>(gridDim.x) * 8;
  for (long long row = static_cast<long long>(blockIdx.x) * 8 + warp; row < n_rows; row += stride) {   // (token, head)
    const int tok = static_cast<int>(row / pd.H);
    // sequence of this token: binary search over cu_seqlens (num_seqs is small)
    int lo = 0, hi = pd.num_seqs - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (pd.seqs[mid].tok_start <= tok) lo = mid; else hi = mid - 1;
    }
    const SeqInfo sq = pd.seqs[lo];
    const int n = tok - sq.tok_start;
    const bool rotate = !pd.no_rope && n < sq.n_video;     // R21: text tokens were not rotated
    int pos[3];
    pos[0] = n / (sq.Hg * sq.Wg); pos[1] = (n / sq.Wg) % sq.Hg; pos[2] = n % sq.Wg;
    const size_t off = static_cast<size_t>(row) * D + d0;      // local fp32 workspace [N, H, D]
    int shard;
    const size_t roff = raw_off(pd.sh, tok, static_cast<int>(row % pd.H), D, shard) + d0;
    const __nv_bfloat16* xraw = shard_base<const __nv_bfloat16>(xraw_s, shard) + roff;
    __nv_bfloat16* out = shard_base<__nv_bfloat16>(out_s, shard) + roff;
    float g[EPL], x[EPL];
    size_t goff = off;
    if (!is_k && pp.gq_blocked) {
      const int gtile = sq.tile_base + n / kTileRows, qr = n % kTileRows;
      goff = (static_cast<size_t>(row % pd.H) * pd.n_tiles_total + gtile) * (kTileRows * D) +
             static_cast<size_t>(d0 >> 5) * (kTileRows * 32) + qr * 32 + ((((d0 & 31) >> 2) ^ (qr & 7)) << 2) + (d0 & 3);
    }
    if constexpr (EPL == 4) {
      const float4 f = *reinterpret_cast<const float4*>(gt + goff);
      g[0] = f.x; g[1] = f.y; g[2] = f.z; g[3] = f.w;
    } else {
      const float2 f = *reinterpret_cast<const float2*>(gt + goff);
      g[0] = f.x; g[1] = f.y;
    }
    load_bf16_row<EPL>(xraw, x);
    if (rotate) {
#pragma unroll
      for (int i = 0; i < EPL; i += 2) {
        const float2 cs = rope_cs(pd.rope, (d0 + i) >> 1, pos);
        const float g0 = g[i], g1 = g[i + 1];
        g[i] = g0 * cs.x + g1 * cs.y;          // rotate by -phi
        g[i + 1] = -g0 * cs.y + g1 * cs.x;
      }
    }
    float y[EPL];
    if (!pd.no_norm) {
      float ss = 0.f, ux = 0.f;
#pragma unroll
      for (int i = 0; i < EPL; ++i) {
        ss += x[i] * x[i];
        ux += gam[i] * g[i] * x[i];
      }
      ss = warp_sum(ss);
      ux = warp_sum(ux);
      const float rinv = rsqrtf(ss * (1.0f / D) + pd.eps);
      const float c = rinv * rinv * rinv * ux * (1.0f / D);
#pragma unroll
      for (int i = 0; i < EPL; ++i) {
        y[i] = rinv * gam[i] * g[i] - c * x[i];
        dgam[i] += g[i] * x[i] * rinv;
      }
    } else {
#pragma unroll
      for (int i = 0; i < EPL; ++i) y[i] = g[i];      // gamma unused: dgamma = 0
    }
    if constexpr (EPL == 4) {
      uint2 u; u.x = pack_bf16x2(y[0], y[1]); u.y = pack_bf16x2(y[2], y[3]);
      *reinterpret_cast<uint2*>(out) = u;
    } else {
      *reinterpret_cast<uint32_t*>(out) = pack_bf16x2(y[0], y[1]);
    }
  }
  if (pp.dgamma_part) {
#pragma unroll
    for (int i = 0; i < EPL; ++i) s_part[warp][d0 + i] = dgam[i];
    __syncthreads();
    if (threadIdx.x < D) {
      float a = 0.f;
#pragma unroll
      for (int w = 0; w < 8; ++w) a += s_part[w][threadIdx.x];
      pp.dgamma_part[(static_cast<size_t>(blockIdx.y) * gridDim.x + blockIdx.x) * D + threadIdx.x] = a;
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

}  // namespace arachne
