// Elementwise pieces of the Q/K load (§8 a1) shared by the prologue (prep.cuh) and the forward's in-kernel variant (fwd.cuh):
// bf16 unpack / 16-bit pack, RoPE table lookup, tile-image addressing, RMSNorm + RoPE of an 8-element chunk.
#pragma once
#include "common.cuh"
#include "sm100.cuh"

namespace arachne {

// sum over the LPR consecutive lanes that share a row
template <int LPR>
__device__ __forceinline__ float seg_sum(float x) {
#pragma unroll
  for (int o = LPR / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

__device__ __forceinline__ void unpack_bf16x8(const uint4& u, float (&x)[8]) {
  x[0] = __uint_as_float(u.x << 16); x[1] = __uint_as_float(u.x & 0xffff0000u);
  x[2] = __uint_as_float(u.y << 16); x[3] = __uint_as_float(u.y & 0xffff0000u);
  x[4] = __uint_as_float(u.z << 16); x[5] = __uint_as_float(u.z & 0xffff0000u);
  x[6] = __uint_as_float(u.w << 16); x[7] = __uint_as_float(u.w & 0xffff0000u);
}
__device__ __forceinline__ uint4 pack8(const float (&y)[8], int fmt) {
  uint4 u;
  if (fmt == FMT_F16) {
    u.x = pack_f16x2(y[0], y[1]); u.y = pack_f16x2(y[2], y[3]); u.z = pack_f16x2(y[4], y[5]); u.w = pack_f16x2(y[6], y[7]);
  } else {
    u.x = pack_bf16x2(y[0], y[1]); u.y = pack_bf16x2(y[2], y[3]); u.z = pack_bf16x2(y[4], y[5]); u.w = pack_bf16x2(y[6], y[7]);
  }
  return u;
}

// (cos, sin) of the 4 RoPE pairs of elements [d0, d0+8) at the token position packed in ti (identity when the token
// is not rotated: text token, R21, or no_rope)
__device__ __forceinline__ void rope_cs4(const RopeDesc& rp, int d0, const TokInfo& ti, bool rotate, float2 (&cs)[4]) {
  const int pos[3] = {static_cast<int>(ti.t_flag & 0x7fffffffu), static_cast<int>(ti.hw >> 16), static_cast<int>(ti.hw & 0xffffu)};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int a = 0, p = (d0 >> 1) + i;
    if (p >= rp.half[0]) { p -= rp.half[0]; a = 1; if (p >= rp.half[1]) { p -= rp.half[1]; a = 2; } }
    cs[i] = rotate ? __ldg(&rp.tab[rp.off[a] + pos[a] * rp.half[a] + p]) : make_float2(1.f, 0.f);
  }
}

// byte offset of the 16-byte chunk holding elements [d0, d0+8) of row r inside a [128][D] tile image
__device__ __forceinline__ uint32_t image_off(int r, int d0) {
  return static_cast<uint32_t>(d0 >> 6) * (kTileRows * 128) + swz_off(r, (d0 & 63) >> 3);
}

// x~ = RoPE(gamma * x * rsqrt(mean(x^2) + eps)) * prescale  (readings R1-R5), in two steps so that the prologue (a row spread
// over D/8 lanes) and the forward's in-kernel variant (a row per thread, fwd.cuh kFusedQ) run the SAME arithmetic in the same
// order: sumsq8 = this 8-element chunk's sum of squares; norm_rope_apply8 = scale by rinv * gamma, rotate, prescale; returns the
// chunk's |x~|^2.
__device__ __forceinline__ float sumsq8(const float (&x)[8]) {
  float ss = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) ss += x[i] * x[i];
  return ss;
}
__device__ __forceinline__ float norm_rope_apply8(float (&x)[8], const float (&gam)[8], const float2 (&cs)[4], bool no_norm, float rinv,
                                                  float prescale) {
  if (!no_norm) {
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] *= rinv * gam[i];
  }
  float nrm = 0.f;
#pragma unroll
  for (int i = 0; i < 8; i += 2) {
    const float2 c = cs[i >> 1];
    const float x0 = x[i], x1 = x[i + 1];
    x[i] = (x0 * c.x - x1 * c.y) * prescale;
    x[i + 1] = (x0 * c.y + x1 * c.x) * prescale;
    nrm += x[i] * x[i] + x[i + 1] * x[i + 1];
  }
  return nrm;
}
// the prologue's form: the row's D/8 lanes each hold one chunk
template <int D>
__device__ __forceinline__ float norm_rope8(float (&x)[8], const float (&gam)[8], const float2 (&cs)[4], bool no_norm,
                                            float eps, float prescale) {
  constexpr int LPR = D / 8;
  float rinv = 1.0f;
  if (!no_norm) rinv = rsqrtf(seg_sum<LPR>(sumsq8(x)) * (1.0f / D) + eps);
  return norm_rope_apply8(x, gam, cs, no_norm, rinv, prescale);
}

}  // namespace arachne
