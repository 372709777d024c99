// Device-visible plan structures shared by all arachne kernels (include/arachne_attn.h is the
// public boundary; this header is internal).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace arachne {

constexpr int kTileRows = 128;   // tokens per tile (query tile == key tile)

// One packed sequence (BASELINE.json north_star: "packed batch ... per-sequence (T,H,W) latent grid").
struct SeqInfo {
  int tok_start;   // cu_seqlens[b]
  int len;         // L_b
  int tile_base;   // index of the sequence's first 128-token tile in the tiled workspace
  int n_tiles;     // ceil(L_b / 128)
  int T, Hg, Wg;   // latent grid; token n -> (n / (Hg*Wg), (n / Wg) % Hg, n % Wg)   (reading R7)
  int qt_lo, qt_n; // query tiles [qt_lo, qt_lo + qt_n) of this sequence are computed by this process: all of them
                   // (0, n_tiles) unless the plan is a context-parallel one (arachne_plan_create_cp)
  int n_video;     // T*Hg*Wg: tokens [0, n_video) are video tokens (rotated); [n_video, len) are text tokens,
                   // normed but NOT rotated (reading R21)
};

// Per-token lookup built by the plan (host): position on the latent grid and place in the tiled workspace, so the
// elementwise kernels need neither integer divisions nor a search over cu_seqlens.
struct TokInfo {
  uint32_t t_flag;   // t (bits 0..30) | bit 31: text token (normed, not rotated: reading R21)
  uint32_t hw;       // h << 16 | w      (grid extents <= 65535, checked by the plan)
  uint32_t blkrow;   // (tile_base + n / 128) * 128 + n % 128: the token's row in the tiled workspace
  uint32_t seq;      // sequence index
};

// One unit of work for the persistent kernels: (sequence, head, 128-token tile of that sequence).
// fwd_kernel reads it as a (pair of) QUERY tile(s), bwd_fused_kernel as a KEY tile.  The host orders the lists
// longest-processing-time-first by (sequence, head) group, tiles of a group adjacent (the deterministic backward list
// interleaves a few groups: arachne_attn.cu); the CTAs take the items dynamically through an atomic counter.
struct WorkItem {
  int seq;
  int head;
  int tile;
  int pad;         // forward items: number of query tiles in the item (1 or 2)
};

// cos/sin tables of the 3D RoPE (readings R4-R6): entry (axis a, position x, pair p) at
// tab[off[a] + x * half[a] + p] = (cos, sin)(x * theta^(-2p/d_a)), computed in fp64 on the host.
struct RopeDesc {
  const float2* tab;
  int off[3];
  int half[3];   // d_a / 2
};

// Raw [tokens, heads, D] tensors may be SHARDED BY TOKEN RANGE across up to kMaxShards buffers (Ulysses sequence
// parallelism): shard r holds the global tokens [start[r], start[r+1]) with ALL
// H_total heads, [n_r, H_total, D]; this process computes heads [head_offset, head_offset + H).  The buffers are any
// device-accessible memory (local, or peer memory mapped over NVLink), so the All-to-All of Ulysses is the prep
// kernel's gather (loads) and the epilogues' scatter (stores) — no staging copy.  n_shards = 1, start = {0, N},
// H_total = H, head_offset = 0 is the plain single-tensor case.
constexpr int kMaxShards = 8;
struct Sharding {
  int n_shards;
  int start[kMaxShards + 1];
  int H_total;
  int head_offset;
};
struct ShardedPtr {
  void* p[kMaxShards];
};
// element offset of (global token tok, local head h, 0) inside its shard; r_out = the shard.  tok_stride = elements between
// consecutive tokens of THIS tensor (H_total * D unless the caller passed a strided Q, K or V: ProblemDesc::in_stride)
__device__ __forceinline__ size_t raw_off(const Sharding& sh, long long tok_stride, int tok, int h, int D, int& r_out) {
  int r = 0;
  if (sh.n_shards > 1) {      // uniform branch: the plain single-tensor case pays nothing
#pragma unroll
    for (int i = 1; i < kMaxShards; ++i)
      if (i < sh.n_shards && tok >= sh.start[i]) r = i;
  }
  r_out = r;
  return static_cast<size_t>(tok - sh.start[r]) * static_cast<size_t>(tok_stride) + static_cast<size_t>(sh.head_offset + h) * D;
}
// t.p[r] with constant indices only (a dynamic index would make ptxas copy the kernel parameter to local memory)
template <typename T>
__device__ __forceinline__ T* shard_base(const ShardedPtr& t, int r) {
  void* b = t.p[0];
  if (r > 0) {
#pragma unroll
    for (int i = 1; i < kMaxShards; ++i)
      if (r == i) b = t.p[i];
  }
  return static_cast<T*>(b);
}
// row of a CONTIGUOUS tensor (everything the library writes, dO, O)
template <typename T>
__device__ __forceinline__ T* raw_row(const Sharding& sh, const ShardedPtr& t, int tok, int h, int D) {
  int r;
  const size_t off = raw_off(sh, static_cast<long long>(sh.H_total) * D, tok, h, D, r);
  return shard_base<T>(t, r) + off;
}

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
constexpr int kTraceMaxCtas = 256;

struct ProblemDesc {
  const SeqInfo* seqs;
  const int* tile_seq;       // [n_tiles_total] tile -> sequence
  const TokInfo* tok_info;   // [N]
  int n_fwd_items;
  const WorkItem* dyn_items;     // [n_items] backward items (key tiles) in the global LPT order, taken dynamically (work_counter)
  const WorkItem* dyn_fwd_items; // [n_fwd_items] forward: pairs of query tiles; .tile = first tile, .pad = tiles in the item (1|2)
  const WorkItem* dyn_fwd_pair_items;  // [n_fwd_pair_items] forward, CTA-pair form: up to FOUR query tiles (.pad = 1..4)
  int n_fwd_pair_items;
  int* work_counter;             // [2] next index into dyn_fwd_items / dyn_items; zeroed by the host before each launch
  unsigned* stats;           // [0] max |q~'|^2, [1] max |k~|^2 (float bits) written by the forward prep kernel.  stats,
                             // work_counter, grp_stats and grp_sk live in the header of the CALLER'S workspace (WsHeader below),
                             // i.e. they are per call: two calls on one plan with different workspaces do not share them
  unsigned* grp_stats;       // backward: [num_seqs * H][4] float bits, (sequence, head) group g: [0] max_i |dO_i|^2, [1] max_j |V_j|^2,
                             // [2] max_j |k~_j|^2 (only without RMSNorm; with it the bound D * max gamma_k^2 is used)
  float* grp_sk;             // backward: [num_seqs * H][4] = (sk, 1/sk, -, -): sk = the power of two dS is multiplied by
                             // before it is rounded to fp16 (bwd_scale_kernel, prep.cuh).  (The fixed-point scale of the
                             // deterministic dq~ reduction is per query ROW: BwdFusedParams::rowqs_t.)
  int n_items;
  int n_tiles_total;
  int num_seqs;
  int N, H;
  float eps;
  float softmax_scale;
  int no_norm, no_rope;
  RopeDesc rope;
  Sharding sh;
  long long in_stride[3];    // token stride (elements) of the raw Q, K, V (arachne_attn_params::q_stride ...; H_total * D if contiguous)
  unsigned long long* cta_trace;   // nullable: [kernel 0 fwd | 1 bwd_fused][gridDim.x][2] globaltimer ns at CTA start / end
  int cp_lo, cp_hi;          // context parallelism: this process owns the QUERY tokens [cp_lo, cp_hi) (0, N otherwise)
};

// Header of every workspace (forward and backward): the per-call mutable words of the kernels.
struct WsHeader {
  unsigned qk_bound[2];      // ProblemDesc::stats
  int work_counter[2];       // ProblemDesc::work_counter ([0] fwd_kernel, [1] bwd_fused_kernel)
  unsigned pad[12];
};
static_assert(sizeof(WsHeader) == 64, "WsHeader");

}  // namespace arachne
