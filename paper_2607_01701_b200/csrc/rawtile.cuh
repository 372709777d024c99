// V and dO tiles read STRAIGHT from the caller's raw [tokens, heads, D] bf16 tensors by the TMA engine (tensor-map
// cp.async.bulk.tensor, SASS UTMALDG): no copy into a tile image in the prologue (§8 a1; SURVEY §7.2 "per-sequence tensor
// maps").  The engine applies the 128-byte swizzle, so the bytes that land in shared memory are exactly the tile image the
// prologue used to write (sm100.cuh): nothing downstream changes.
//
// Tensor map: 3-D (head_dim elements, heads, tokens), box = 64 elements x 1 head x R tokens; one box = one 64-element block
// [R rows x 128 B] of a tile.  Two maps per tensor: R = 128 (whole tiles) and R = 8 (the ragged last tile of a sequence).
// A tile never holds rows of another sequence: of a last tile with `valid` < 128 rows
//   * rows [0, valid & ~7) come as 8-row boxes,
//   * rows [valid & ~7, valid) are copied by the producer warp (16-byte loads, swizzled stores),
//   * rows [valid, 128) are zeroed by the producer warp,
// the generic-proxy stores being fenced (fence.proxy.async) before the tile's mbarrier can complete.  So the rows after a
// sequence's end are exact zeros as in the image path, whatever the neighbouring sequence holds (NaN included).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "sm100.cuh"

namespace arachne {

struct RawMaps {
  CUtensorMap tile;    // box 64 x 1 x 128
  CUtensorMap rows8;   // box 64 x 1 x 8
};

// the same tensor for the generic-proxy part of a ragged tile (and "is the raw path on": base != nullptr)
struct RawTensor {
  const __nv_bfloat16* base;
  long long tok_stride;    // elements between consecutive tokens
  int head0;               // first head of this process inside the tensor (Sharding::head_offset)
};

// Whole producer warp.  Prepares the rows of tile (head, tokens [tok0, tok0 + valid)) that the TMA engine does not write
// and returns the number of bytes it WILL write (the transaction count to expect on the tile's mbarrier).
template <int D>
__device__ __forceinline__ uint32_t raw_tile_stage(uint8_t* dst, const RawTensor& rt, int head, int tok0, int valid, int lane) {
  if (valid >= kTileRows) return kTileRows * D * 2;
  constexpr int CPR = D / 8;                      // 16-byte chunks per row
  const int r8 = valid & ~7;
  // rows [r8, valid): copy
  const __nv_bfloat16* src = rt.base + static_cast<long long>(tok0) * rt.tok_stride + static_cast<long long>(rt.head0 + head) * D;
  for (int i = lane; i < (valid - r8) * CPR; i += 32) {
    const int r = r8 + i / CPR, ch = i % CPR;
    const uint4 u = *reinterpret_cast<const uint4*>(src + static_cast<long long>(r) * rt.tok_stride + ch * 8);
    *reinterpret_cast<uint4*>(dst + (ch >> 3) * (kTileRows * 128) + swz_off(r, ch & 7)) = u;
  }
  // rows [valid, 128): zero (whole rows, so the swizzle does not matter)
  const uint4 z = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
  for (int c = 0; c < D / 64; ++c)
    for (int i = lane; i < (kTileRows - valid) * 8; i += 32)
      *reinterpret_cast<uint4*>(dst + c * (kTileRows * 128) + valid * 128 + i * 16) = z;
  fence_proxy_async_smem();
  __syncwarp();
  return static_cast<uint32_t>(r8) * D * 2;
}

// One lane, after the transaction count has been put on `bar`.
template <int D>
__device__ __forceinline__ void raw_tile_issue(uint8_t* dst, const RawMaps& m, const RawTensor& rt, int head, int tok0, int valid,
                                               uint64_t* bar) {
  const int h = rt.head0 + head;
  if (valid >= kTileRows) {
#pragma unroll
    for (int c = 0; c < D / 64; ++c) tma_load_3d(dst + c * (kTileRows * 128), &m.tile, 64 * c, h, tok0, bar);
  } else {
    for (int r = 0; r + 8 <= valid; r += 8)
#pragma unroll
      for (int c = 0; c < D / 64; ++c) tma_load_3d(dst + c * (kTileRows * 128) + r * 128, &m.rows8, 64 * c, h, tok0 + r, bar);
  }
}

// Multicast form (cluster of 2, D = 128): CTA `rank` fetches the 64-element block `rank` of the tile and multicasts it into
// both CTAs' slots; each CTA has staged the generic-proxy rows of a ragged tile itself.
template <int D>
__device__ __forceinline__ void raw_tile_issue_mc(uint8_t* dst, const RawMaps& m, const RawTensor& rt, int head, int tok0, int valid,
                                                  uint64_t* bar, uint32_t rank) {
  static_assert(D == 128, "two 64-element blocks, one per CTA of the cluster");
  const int h = rt.head0 + head, c = static_cast<int>(rank);
  if (valid >= kTileRows) {
    tma_load_3d_mc(dst + c * (kTileRows * 128), &m.tile, 64 * c, h, tok0, bar, 3);
  } else {
    for (int r = 0; r + 8 <= valid; r += 8) tma_load_3d_mc(dst + c * (kTileRows * 128) + r * 128, &m.rows8, 64 * c, h, tok0 + r, bar, 3);
  }
}

}  // namespace arachne
