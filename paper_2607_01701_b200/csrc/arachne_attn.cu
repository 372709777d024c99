// libarachne_attn.so — C ABI (include/arachne_attn.h) over the sm_100a kernels.
// Host side: validation, the plan (tile work list in LPT order, RoPE tables), workspace carving
// and kernel launches.  No torch types, no hidden allocation or synchronisation in fwd/bwd.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/arachne_attn.h"
#include "bwd_fused.cuh"
#include "common.cuh"
#include "fwd.cuh"
#include "prep.cuh"
#include "rawtile.cuh"

using namespace arachne;

namespace {

thread_local std::string g_last_error;

int cuda_fail(cudaError_t e, const char* what) {
  g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
  return ARACHNE_ERR_CUDA;
}
#define ARACHNE_CUDA(call)                                  \
  do {                                                      \
    cudaError_t e__ = (call);                               \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call);   \
  } while (0)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
bool misaligned(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

}  // namespace

struct arachne_host_ctx;
static void arachne_host_ctx_free(arachne_host_ctx*);

struct arachne_plan {
  arachne_attn_params p;
  std::vector<int32_t> cu;
  std::vector<SeqInfo> seqs;
  int n_tiles_total = 0;
  int n_items = 0;
  int num_sms = 0;
  int device = 0;
  mutable struct arachne_host_ctx* host = nullptr;   // lazily created by the *_host calls (device buffers, streams)
  int cp_rank = -1;   // >= 0: context-parallel plan (arachne_plan_create_cp), this process owns the queries of shard cp_rank
  Sharding sh{};   // token-range sharding of the raw tensors (1 shard = plain tensors)
  int n_groups = 0;        // num_seqs * num_heads: (sequence, head) groups (dS scaling tables in the workspace header)
  size_t hdr_bytes = 0;    // WsHeader + group tables at the start of every workspace
  unsigned* d_envelope = nullptr;   // sticky: float bits of the largest out-of-envelope logit bound seen (arachne_plan_logit_status)
  float bound_limit = 0.f; // forward: logit bound (log2 units) above which a launch without ARACHNE_FLAG_WIDE_LOGITS is flagged
  // device arrays (owned)
  SeqInfo* d_seqs = nullptr;
  int* d_tile_seq = nullptr;
  TokInfo* d_tok_info = nullptr;
  WorkItem* d_dyn_items = nullptr;      // the global LPT-ordered lists (dynamic distribution in fwd_kernel / bwd_fused_kernel)
  WorkItem* d_dyn_fwd_items = nullptr;
  int n_ctas = 0, n_fwd_ctas = 0;
  int n_fwd_items = 0;
  WorkItem* d_dyn_fwd_pair_items = nullptr;   // forward, CTA-pair form: items of up to four query tiles
  int n_fwd_pair_items = 0, n_fwd_pair_ctas = 0;
  bool fwd_pairs = false;               // D = 128 and ARACHNE_FLAG_FWD_CTA_PAIRS: fwd_pair_kernel
  bool fwd_mcast = false;               // D = 128 and ARACHNE_FLAG_FWD_MULTICAST: fwd_mc_kernel
  bool fwd_fused_q = false;             // ARACHNE_FLAG_FWD_FUSED_Q: fwd_kernel normalises its own raw query tiles (A/B of a1)
  bool raw_fwd = false, raw_bwd = false;   // V (fwd) / V and dO (bwd) tiles are read from the raw tensors by tensor-map TMA
                                           // (rawtile.cuh) instead of being copied into tile images by the prologue
  int n_img_fwd = 3, n_img_bwd = 4;        // tile-image regions in the forward / backward workspace
  unsigned long long* d_cta_trace = nullptr;   // [2][kTraceMaxCtas][2] globaltimer ns (arachne_plan_cta_times)
  float2* d_rope = nullptr;
  ProblemDesc pd{};
  // workspace layout
  size_t tile_bytes = 0, img_bytes = 0, rowvec_bytes = 0, grad_bytes = 0, gradblk_bytes = 0, dgpart_bytes = 0;
  int post_blocks = 0;   // post_kernel grid.x (grid-stride over groups of tokens); fixes the dgamma summation order
  // optional per-kernel timing (arachne_plan_enable_profiling): ring of kProfSlots calls per pass,
  // kernels+1 events per call, recorded on the caller's stream (no synchronisation).
  static constexpr int kProfSlots = 32;
  static constexpr int kMaxKernels = 3;
  bool profiling = false;
  mutable long long prof_calls[2] = {0, 0};
  cudaEvent_t prof_ev[2][kProfSlots][kMaxKernels + 1] = {};
};

static int plan_create_impl(arachne_plan** out, const arachne_attn_params* params, const int32_t* cu, const int32_t* grids,
                            const int32_t* text_lens, int32_t num_shards, const int32_t* shard_starts,
                            int32_t total_heads, int32_t head_offset, int cp_rank);

namespace {

template <int D>
int configure_kernels() {
  ARACHNE_CUDA(cudaFuncSetAttribute(fwd_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, FwdCfg<D>::kSmemBytes));
  ARACHNE_CUDA(cudaFuncSetAttribute(fwd_kernel<D, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, FwdCfg<D>::kSmemBytes));
  if constexpr (D == 128)
    ARACHNE_CUDA(cudaFuncSetAttribute(fwd_pair_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, FwdCfg<D, kFwdPair>::kSmemBytes));
  if constexpr (D == 128)
    ARACHNE_CUDA(cudaFuncSetAttribute(fwd_mc_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, FwdCfg<D, kFwdMcast>::kSmemBytes));
  ARACHNE_CUDA(cudaFuncSetAttribute(bwd_fused_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, BwdFusedCfg<D>::kSmemBytes));
  return ARACHNE_OK;
}

struct FwdWs { uint8_t *qt, *kt, *vt; };
struct BwdWs { uint8_t *qt, *kt, *vt, *dot; float *lse2_t, *delta_t, *rowqs_t, *gq_t, *gk_t; };

size_t fwd_ws_bytes(const arachne_plan* pl) { return pl->hdr_bytes + pl->n_img_fwd * pl->img_bytes; }
// (3 row vectors: lse2, delta and the per-row fixed-point scales of the deterministic dq~ reduction)
size_t bwd_ws_bytes(const arachne_plan* pl) { return pl->hdr_bytes + pl->n_img_bwd * pl->img_bytes + 3 * pl->rowvec_bytes + pl->grad_bytes + pl->gradblk_bytes + pl->dgpart_bytes; }

// Tensor maps over a raw [tokens, H_total, D] bf16 tensor (rawtile.cuh): encoded on the host per call (the base pointer is a
// call argument), ~1 us each, passed to the kernel as __grid_constant__ parameters.  cuTensorMapEncodeTiled is taken from
// the driver at run time (no link-time dependency on libcuda).
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess || qr != cudaDriverEntryPointSuccess)
      p = nullptr;
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}
int make_raw_maps(const arachne_plan* pl, const void* base, long long tok_stride, RawMaps* out, RawTensor* rt) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) { g_last_error = "cuTensorMapEncodeTiled not available from the driver"; return ARACHNE_ERR_CUDA; }
  const cuuint64_t D = static_cast<cuuint64_t>(pl->p.head_dim), Ht = static_cast<cuuint64_t>(pl->sh.H_total);
  const cuuint64_t dims[3] = {D, Ht, static_cast<cuuint64_t>(pl->p.total_tokens)};
  const cuuint64_t strides[2] = {D * 2, static_cast<cuuint64_t>(tok_stride) * 2};      // bytes, dims 1 (heads) and 2 (tokens)
  const cuuint32_t estr[3] = {1, 1, 1};
  for (int i = 0; i < 2; ++i) {
    const cuuint32_t box[3] = {64, 1, i == 0 ? static_cast<cuuint32_t>(kTileRows) : 8u};
    const CUresult r = enc(i == 0 ? &out->tile : &out->rows8, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims,
                           strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { g_last_error = "cuTensorMapEncodeTiled failed (" + std::to_string(static_cast<int>(r)) + ")"; return ARACHNE_ERR_CUDA; }
  }
  rt->base = static_cast<const __nv_bfloat16*>(base);
  rt->tok_stride = tok_stride;
  rt->head0 = pl->sh.head_offset;
  return ARACHNE_OK;
}

// The first hdr_bytes of every workspace hold the per-call mutable words of the kernels (WsHeader: logit bound, dynamic
// work counters) and, for the backward, the per-(sequence, head) dS-scaling tables: the plan itself carries no per-launch
// state, so concurrent calls on one plan are safe as long as each has its own workspace.
ProblemDesc per_call_desc(const arachne_plan* pl, void* ws) {
  ProblemDesc pd = pl->pd;
  uint8_t* w = static_cast<uint8_t*>(ws);
  WsHeader* hdr = reinterpret_cast<WsHeader*>(w);
  pd.stats = hdr->qk_bound;
  pd.work_counter = hdr->work_counter;
  pd.grp_stats = reinterpret_cast<unsigned*>(w + sizeof(WsHeader));
  pd.grp_sk = reinterpret_cast<float*>(w + sizeof(WsHeader) + static_cast<size_t>(pl->n_groups) * 16);
  return pd;
}

inline void prof_mark(const arachne_plan* pl, int pass, int idx, cudaStream_t st) {
  if (!pl->profiling) return;
  const int slot = static_cast<int>(pl->prof_calls[pass] % arachne_plan::kProfSlots);
  cudaEventRecord(pl->prof_ev[pass][slot][idx], st);
}

template <int D>
int launch_fwd(const arachne_plan* pl, const ShardedPtr& q, const ShardedPtr& k, const ShardedPtr& v, const float* gq,
               const float* gk, const ShardedPtr& o, float* lse, void* ws, cudaStream_t st) {
  uint8_t* w = static_cast<uint8_t*>(ws) + pl->hdr_bytes;
  FwdWs f{w, w + pl->img_bytes, pl->raw_fwd ? nullptr : w + 2 * pl->img_bytes};
  const ProblemDesc pd = per_call_desc(pl, ws);
  RawMaps vmaps{};
  RawTensor v_raw{};
  if (pl->raw_fwd) {
    const int rc = make_raw_maps(pl, v.p[0], pl->pd.in_stride[2], &vmaps, &v_raw);
    if (rc != ARACHNE_OK) return rc;
  }
  PrepParams pp{};
  pp.q = q; pp.k = k; pp.v = v;
  pp.gamma_q = gq; pp.gamma_k = gk;
  pp.qt = f.qt; pp.kt = f.kt; pp.vt = f.vt;
  pp.q_prescale = pl->p.softmax_scale * 1.4426950408889634f;   // S leaves the tensor core in the exp2 domain
  pp.stats = pd.stats;
  pp.skip_q = pl->fwd_fused_q ? 1 : 0;
  RawMaps qmaps{};
  RawTensor q_raw{};
  if (pl->fwd_fused_q) {
    const int rc = make_raw_maps(pl, q.p[0], pl->pd.in_stride[0], &qmaps, &q_raw);
    if (rc != ARACHNE_OK) return rc;
  }
  prof_mark(pl, 0, 0, st);
  ARACHNE_CUDA(cudaMemsetAsync(ws, 0, sizeof(WsHeader), st));
  if (pl->raw_fwd) prep_kernel<D, false, false><<<dim3(pl->n_tiles_total, pl->p.num_heads), 256, 0, st>>>(pd, pp);
  else prep_kernel<D, false, true><<<dim3(pl->n_tiles_total, pl->p.num_heads), 256, 0, st>>>(pd, pp);
  ARACHNE_CUDA(cudaGetLastError());
  prof_mark(pl, 0, 1, st);
  FwdParams fp{f.qt, f.kt, f.vt, v_raw, q_raw, gq, pp.q_prescale, o, lse, pl->d_envelope, pl->bound_limit};
  if constexpr (D == 128) {
    if (pl->fwd_pairs) {      // CTA-pair form (cluster of 2, cta_group::2): grid = 2 CTAs per pair
      if (pl->n_fwd_pair_ctas > 0)
        fwd_pair_kernel<D><<<pl->n_fwd_pair_ctas, FwdCfg<D, kFwdPair>::kThreads, FwdCfg<D, kFwdPair>::kSmemBytes, st>>>(pd, fp, vmaps);
      ARACHNE_CUDA(cudaGetLastError());
      prof_mark(pl, 0, 2, st);
      if (pl->profiling) pl->prof_calls[0]++;
      return ARACHNE_OK;
    }
  }
  if constexpr (D == 128) {
    if (pl->fwd_mcast) {      // multicast form (cluster of 2 sharing the K^/V stream): grid = 2 CTAs per cluster
      if (pl->n_fwd_pair_ctas > 0)
        fwd_mc_kernel<D><<<pl->n_fwd_pair_ctas, FwdCfg<D, kFwdMcast>::kThreads, FwdCfg<D, kFwdMcast>::kSmemBytes, st>>>(pd, fp, vmaps);
      ARACHNE_CUDA(cudaGetLastError());
      prof_mark(pl, 0, 2, st);
      if (pl->profiling) pl->prof_calls[0]++;
      return ARACHNE_OK;
    }
  }
  const int grid = pl->n_fwd_ctas;
  if (grid > 0) {
    if (pl->fwd_fused_q) fwd_kernel<D, true><<<grid, FwdCfg<D>::kThreads, FwdCfg<D>::kSmemBytes, st>>>(pd, fp, vmaps, qmaps);
    else fwd_kernel<D><<<grid, FwdCfg<D>::kThreads, FwdCfg<D>::kSmemBytes, st>>>(pd, fp, vmaps, qmaps);
  }   // (a CP rank may own no queries)
  ARACHNE_CUDA(cudaGetLastError());
  prof_mark(pl, 0, 2, st);
  if (pl->profiling) pl->prof_calls[0]++;
  return ARACHNE_OK;
}

template <int D>
int launch_bwd(const arachne_plan* pl, const ShardedPtr& q, const ShardedPtr& k, const ShardedPtr& v, const float* gq,
               const float* gk, const ShardedPtr& o, const float* lse, const ShardedPtr& d_o, const ShardedPtr& dq,
               const ShardedPtr& dk, const ShardedPtr& dv, float* dgq, float* dgk, void* ws, cudaStream_t st,
               float* cp_gk = nullptr, float* cp_gv = nullptr) {
  // cp_gk / cp_gv (context parallelism, phase 1): dk~ and dV leave as fp32 PARTIALS in these [N,H,D] buffers, only dQ is
  // finished here (for this rank's query rows); arachne_cp_reduce finishes dK, dV.
  const bool cp = cp_gk != nullptr;
  uint8_t* w = static_cast<uint8_t*>(ws) + pl->hdr_bytes;
  const ProblemDesc pd = per_call_desc(pl, ws);
  BwdWs b{};
  b.qt = w; w += pl->img_bytes;
  b.kt = w; w += pl->img_bytes;
  if (!pl->raw_bwd) {
    b.vt = w; w += pl->img_bytes;
    b.dot = w; w += pl->img_bytes;
  }
  RawMaps vmaps{}, domaps{};
  RawTensor v_raw{}, do_raw{};
  if (pl->raw_bwd) {
    int rc;
    if ((rc = make_raw_maps(pl, v.p[0], pl->pd.in_stride[2], &vmaps, &v_raw)) != ARACHNE_OK ||
        (rc = make_raw_maps(pl, d_o.p[0], static_cast<long long>(pl->sh.H_total) * pl->p.head_dim, &domaps, &do_raw)) != ARACHNE_OK)
      return rc;
  }
  b.lse2_t = reinterpret_cast<float*>(w); w += pl->rowvec_bytes;
  b.delta_t = reinterpret_cast<float*>(w); w += pl->rowvec_bytes;
  b.rowqs_t = reinterpret_cast<float*>(w); w += pl->rowvec_bytes;
  b.gk_t = reinterpret_cast<float*>(w); w += pl->grad_bytes;
  b.gq_t = reinterpret_cast<float*>(w); w += pl->gradblk_bytes;     // gradblk_bytes >= grad_bytes: either layout fits
  float* dgpart = (dgq || dgk) ? reinterpret_cast<float*>(w) : nullptr;
  if (cp) b.gk_t = cp_gk;
  const bool deterministic = (pl->p.flags & ARACHNE_FLAG_DETERMINISTIC) != 0;
  PrepParams pp{};
  pp.q = q; pp.k = k; pp.v = v; pp.d_o = d_o; pp.o = o; pp.lse = lse;
  pp.gamma_q = gq; pp.gamma_k = gk;
  pp.qt = b.qt; pp.kt = b.kt; pp.vt = b.vt; pp.dot = b.dot; pp.lse2_t = b.lse2_t; pp.delta_t = b.delta_t;
  pp.q_prescale = pl->p.softmax_scale * 1.4426950408889634f;   // the forward's operand images, bit for bit
  pp.gq_zero = b.gq_t;
  pp.rowqs_t = deterministic ? b.rowqs_t : nullptr;
  prof_mark(pl, 1, 0, st);
  ARACHNE_CUDA(cudaMemsetAsync(ws, 0, sizeof(WsHeader) + static_cast<size_t>(pl->n_groups) * 16, st));   // header, group maxima
  if (pl->raw_bwd) prep_kernel<D, true, false><<<dim3(pl->n_tiles_total, pl->p.num_heads), 256, 0, st>>>(pd, pp);
  else prep_kernel<D, true, true><<<dim3(pl->n_tiles_total, pl->p.num_heads), 256, 0, st>>>(pd, pp);
  ARACHNE_CUDA(cudaGetLastError());
  bwd_scale_kernel<<<dim3(pl->n_tiles_total, pl->p.num_heads), 128, 0, st>>>(pd, b.delta_t, gk, D, pp.rowqs_t);
  ARACHNE_CUDA(cudaGetLastError());
  prof_mark(pl, 1, 1, st);
  const int grid = pl->n_ctas;
  {
    // fused single-pass (5 GEMM) kernel: dQ~ partial tiles reduce-added at L2 — fp32 in arrival order by default, int32
    // fixed point (order-independent, bit-reproducible) with ARACHNE_FLAG_DETERMINISTIC
    BwdFusedParams bp{b.qt, b.kt, b.vt, b.dot, v_raw, do_raw, b.lse2_t, b.delta_t, b.gq_t, b.gk_t, dv, cp_gv, deterministic ? 1 : 0, b.rowqs_t};
    if (grid > 0) bwd_fused_kernel<D><<<grid, BwdFusedCfg<D>::kThreads, BwdFusedCfg<D>::kSmemBytes, st>>>(pd, bp, vmaps, domaps);
    ARACHNE_CUDA(cudaGetLastError());
    prof_mark(pl, 1, 2, st);
  }
  PostParams po{b.gq_t, 1, deterministic ? 1 : 0, b.gk_t, q, k, gq, gk, dq, dk, cp ? 1 : 0, pl->pd.cp_lo, pl->pd.cp_hi, dgpart, b.rowqs_t};
  post_kernel<D><<<dim3(pl->post_blocks, cp ? 1 : 2), 256, 0, st>>>(pd, po);
  ARACHNE_CUDA(cudaGetLastError());
  if (dgpart) {
    dgamma_reduce_kernel<D><<<2, 256, 0, st>>>(dgpart, pl->post_blocks, dgq, dgk);
    ARACHNE_CUDA(cudaGetLastError());
  }
  prof_mark(pl, 1, 3, st);
  if (pl->profiling) pl->prof_calls[1]++;
  return ARACHNE_OK;
}

}  // namespace

extern "C" {

const char* arachne_status_string(int s) {
  switch (s) {
    case ARACHNE_OK: return "ok";
    case ARACHNE_ERR_NULL_POINTER: return "null pointer";
    case ARACHNE_ERR_BAD_HEAD_DIM: return "head_dim must be 64 or 128";
    case ARACHNE_ERR_BAD_ROPE_DIMS: return "rope_dims must be even, non-negative and sum to head_dim";
    case ARACHNE_ERR_BAD_CU_SEQLENS: return "cu_seqlens must start at 0 and be strictly increasing";
    case ARACHNE_ERR_GRID_MISMATCH: return "T*Hg*Wg != sequence length";
    case ARACHNE_ERR_TOTAL_TOKENS: return "cu_seqlens[num_seqs] != total_tokens";
    case ARACHNE_ERR_MISALIGNED: return "pointer not 16-byte aligned";
    case ARACHNE_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case ARACHNE_ERR_BAD_ARCH: return "device is not compute capability 10.x (B200 / sm_100a required)";
    case ARACHNE_ERR_CUDA: return "CUDA runtime error";
    case ARACHNE_ERR_BAD_SHAPE: return "bad shape";
    case ARACHNE_ERR_BAD_PARAM: return "bad parameter";
    case ARACHNE_ERR_BAD_SHARDING: return "bad sharding (1..8 shards, starts 0..N non-decreasing, head_offset + num_heads <= total_heads)";
    case ARACHNE_ERR_LOGIT_RANGE: return "logit range outside the verified envelope (softmax_scale*sqrt(D)*|gamma_q|inf*|gamma_k|inf > 1): pass ARACHNE_FLAG_WIDE_LOGITS";
    case ARACHNE_ERR_BUILTIN_SCRATCH: return "packing too large for the built-in scratch of arachne_varlen_attn_fwd_noalloc (32 MiB): use arachne_varlen_attn_fwd with a workspace";
    default: return "unknown status";
  }
}

const char* arachne_last_error_message(void) { return g_last_error.c_str(); }

int arachne_abi_version(void) { return ARACHNE_ABI_VERSION; }
size_t arachne_attn_params_size(void) { return sizeof(arachne_attn_params); }

int arachne_plan_create(arachne_plan** out, const arachne_attn_params* params, const int32_t* cu, const int32_t* grids) {
  return arachne_plan_create_joint(out, params, cu, grids, nullptr);
}

int arachne_plan_create_joint(arachne_plan** out, const arachne_attn_params* params, const int32_t* cu, const int32_t* grids,
                              const int32_t* text_lens) {
  return arachne_plan_create_sharded(out, params, cu, grids, text_lens, 1, nullptr, params ? params->num_heads : 0, 0);
}

int arachne_plan_create_sharded(arachne_plan** out, const arachne_attn_params* params, const int32_t* cu, const int32_t* grids,
                                const int32_t* text_lens, int32_t num_shards, const int32_t* shard_starts,
                                int32_t total_heads, int32_t head_offset) {
  return plan_create_impl(out, params, cu, grids, text_lens, num_shards, shard_starts, total_heads, head_offset, -1);
}

int arachne_plan_create_cp(arachne_plan** out, const arachne_attn_params* params, const int32_t* cu, const int32_t* grids,
                           const int32_t* text_lens, int32_t num_shards, const int32_t* shard_starts, int32_t rank) {
  if (!params) return ARACHNE_ERR_NULL_POINTER;
  if (rank < 0 || rank >= num_shards) return ARACHNE_ERR_BAD_SHARDING;
  return plan_create_impl(out, params, cu, grids, text_lens, num_shards, shard_starts, params->num_heads, 0, rank);
}

}  // extern "C"
static int plan_create_impl(arachne_plan** out, const arachne_attn_params* params, const int32_t* cu, const int32_t* grids,
                            const int32_t* text_lens, int32_t num_shards, const int32_t* shard_starts,
                            int32_t total_heads, int32_t head_offset, int cp_rank) {
  if (!out || !params || !cu || !grids) return ARACHNE_ERR_NULL_POINTER;
  if (num_shards < 1 || num_shards > kMaxShards || (num_shards > 1 && !shard_starts)) return ARACHNE_ERR_BAD_SHARDING;
  if (head_offset < 0 || params->num_heads <= 0 || static_cast<long long>(head_offset) + params->num_heads > total_heads)
    return ARACHNE_ERR_BAD_SHARDING;
  if (shard_starts) {
    if (shard_starts[0] != 0 || shard_starts[num_shards] != params->total_tokens) return ARACHNE_ERR_BAD_SHARDING;
    for (int r = 0; r < num_shards; ++r)
      if (shard_starts[r + 1] < shard_starts[r]) return ARACHNE_ERR_BAD_SHARDING;      // empty shards are allowed
  }
  *out = nullptr;
  const arachne_attn_params& p = *params;
  if (p.head_dim != 64 && p.head_dim != 128) return ARACHNE_ERR_BAD_HEAD_DIM;
  if (p.num_seqs <= 0 || p.num_heads <= 0 || p.total_tokens <= 0 || p.num_heads > 65535) return ARACHNE_ERR_BAD_SHAPE;
  // 32-bit row / item indices on the device: (tokens + one tile of padding per sequence) x heads must stay below 2^31
  if ((static_cast<long long>(p.total_tokens) + 128LL * p.num_seqs) * p.num_heads >= (1LL << 31)) return ARACHNE_ERR_BAD_SHAPE;
  int rsum = 0;
  for (int a = 0; a < 3; ++a) {
    if (p.rope_dims[a] < 0 || (p.rope_dims[a] & 1)) return ARACHNE_ERR_BAD_ROPE_DIMS;
    rsum += p.rope_dims[a];
  }
  if (rsum != p.head_dim) return ARACHNE_ERR_BAD_ROPE_DIMS;
  if (!(p.rope_theta > 0.f) || !std::isfinite(p.rope_theta) || !(p.rms_eps >= 0.f) || !std::isfinite(p.rms_eps) ||
      !(p.softmax_scale >= 0.f) || !std::isfinite(p.softmax_scale) || (p.flags & ~255))
    return ARACHNE_ERR_BAD_PARAM;
  {
    // envelope (reading R19): an explicit softmax_scale above 1/sqrt(D) widens the logits beyond what the gates are claimed for
    const float sc = p.softmax_scale == 0.f ? 1.0f / std::sqrt(static_cast<float>(p.head_dim)) : p.softmax_scale;
    if (sc * std::sqrt(static_cast<float>(p.head_dim)) > 1.0001f && !(p.flags & (ARACHNE_FLAG_WIDE_LOGITS | ARACHNE_FLAG_NO_NORM)))
      return ARACHNE_ERR_LOGIT_RANGE;
  }
  {
    // token strides of Q, K, V: one-shard plans over a tensor of exactly num_heads heads; 16-byte rows; no overlap
    const long long hd = static_cast<long long>(p.num_heads) * p.head_dim;
    for (long long sx : {static_cast<long long>(p.q_stride), static_cast<long long>(p.k_stride), static_cast<long long>(p.v_stride)}) {
      if (sx == 0) continue;
      if (num_shards != 1 || total_heads != p.num_heads || sx < hd || (sx % 8) != 0) return ARACHNE_ERR_BAD_PARAM;
    }
  }
  if (cu[0] != 0) return ARACHNE_ERR_BAD_CU_SEQLENS;
  for (int b = 0; b < p.num_seqs; ++b)
    if (cu[b + 1] <= cu[b]) return ARACHNE_ERR_BAD_CU_SEQLENS;          // R16: L_b >= 1
  if (cu[p.num_seqs] != p.total_tokens) return ARACHNE_ERR_TOTAL_TOKENS;
  for (int b = 0; b < p.num_seqs; ++b) {
    const int32_t* g = grids + 3 * b;
    if (g[0] <= 0 || g[1] <= 0 || g[2] <= 0) return ARACHNE_ERR_GRID_MISMATCH;
    if (g[1] > 65535 || g[2] > 65535) return ARACHNE_ERR_BAD_SHAPE;      // TokInfo packs h, w into 16 bits each
    const long long nt = text_lens ? text_lens[b] : 0;      // R21: trailing text tokens
    if (nt < 0) return ARACHNE_ERR_BAD_SHAPE;
    if (static_cast<long long>(g[0]) * g[1] * g[2] + nt != static_cast<long long>(cu[b + 1] - cu[b])) return ARACHNE_ERR_GRID_MISMATCH;
  }
  int dev = 0;
  cudaDeviceProp prop{};
  ARACHNE_CUDA(cudaGetDevice(&dev));
  ARACHNE_CUDA(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) return ARACHNE_ERR_BAD_ARCH;

  arachne_plan* pl = new (std::nothrow) arachne_plan();
  if (!pl) { g_last_error = "out of host memory"; return ARACHNE_ERR_CUDA; }
  pl->p = p;
  if (pl->p.softmax_scale == 0.f) pl->p.softmax_scale = 1.0f / std::sqrt(static_cast<float>(p.head_dim));   // R8
  pl->device = dev;
  pl->num_sms = prop.multiProcessorCount;
  pl->cu.assign(cu, cu + p.num_seqs + 1);
  int tile_base = 0, ext[3] = {1, 1, 1};
  for (int b = 0; b < p.num_seqs; ++b) {
    SeqInfo s{};
    s.tok_start = cu[b]; s.len = cu[b + 1] - cu[b];
    s.tile_base = tile_base; s.n_tiles = (s.len + kTileRows - 1) / kTileRows;
    s.T = grids[3 * b]; s.Hg = grids[3 * b + 1]; s.Wg = grids[3 * b + 2];
    s.n_video = s.T * s.Hg * s.Wg;
    s.qt_lo = 0; s.qt_n = s.n_tiles;
    if (cp_rank >= 0) {      // context parallelism: only the query tiles that hold tokens of [starts[rank], starts[rank+1])
      const int lo = std::max(shard_starts ? shard_starts[cp_rank] : 0, s.tok_start);
      const int hi = std::min(shard_starts ? shard_starts[cp_rank + 1] : p.total_tokens, s.tok_start + s.len);
      s.qt_lo = lo < hi ? (lo - s.tok_start) / kTileRows : 0;
      s.qt_n = lo < hi ? (hi - 1 - s.tok_start) / kTileRows + 1 - s.qt_lo : 0;
    }
    tile_base += s.n_tiles;
    for (int a = 0; a < 3; ++a) ext[a] = std::max(ext[a], grids[3 * b + a]);
    pl->seqs.push_back(s);
  }
  pl->n_tiles_total = tile_base;
  pl->cp_rank = cp_rank;
  std::vector<int> tile_seq(pl->n_tiles_total);
  for (int b = 0; b < p.num_seqs; ++b)
    for (int t = 0; t < pl->seqs[b].n_tiles; ++t) tile_seq[pl->seqs[b].tile_base + t] = b;
  // Work list: (sequence, head) groups in longest-processing-time-first order (a tile of sequence b
  // costs n_tiles_b inner iterations), tiles of one group adjacent so that CTAs running side by
  // side stream the same K/V (or Q/dO) tiles through L2.
  std::vector<int> order(p.num_seqs);
  for (int b = 0; b < p.num_seqs; ++b) order[b] = b;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return pl->seqs[a].n_tiles > pl->seqs[b].n_tiles; });
  std::vector<WorkItem> items;
  for (int b : order)
    for (int h = 0; h < p.num_heads; ++h)
      for (int t = 0; t < pl->seqs[b].n_tiles && pl->seqs[b].qt_n > 0; ++t) items.push_back(WorkItem{b, h, t, 0});
  // forward items: pairs of adjacent query tiles (two tiles ping-pong on the tensor pipe), same group order
  std::vector<WorkItem> fwd_items;
  for (int b : order)
    for (int h = 0; h < p.num_heads; ++h)
      for (int t = pl->seqs[b].qt_lo; t < pl->seqs[b].qt_lo + pl->seqs[b].qt_n; t += 2)
        fwd_items.push_back(WorkItem{b, h, t, std::min(2, pl->seqs[b].qt_lo + pl->seqs[b].qt_n - t)});
  // CTA-pair forward: items of up to FOUR adjacent query tiles (two per CTA of the pair), same group order
  std::vector<WorkItem> fwd_pair_items;
  for (int b : order)
    for (int h = 0; h < p.num_heads; ++h)
      for (int t = pl->seqs[b].qt_lo; t < pl->seqs[b].qt_lo + pl->seqs[b].qt_n; t += 4)
        fwd_pair_items.push_back(WorkItem{b, h, t, std::min(4, pl->seqs[b].qt_lo + pl->seqs[b].qt_n - t)});
  pl->n_fwd_pair_items = static_cast<int>(fwd_pair_items.size());
  pl->n_fwd_pair_ctas = 2 * std::min(pl->num_sms / 2, pl->n_fwd_pair_items);
  pl->fwd_pairs = p.head_dim == 128 && (p.flags & ARACHNE_FLAG_FWD_CTA_PAIRS) != 0;
  pl->fwd_mcast = p.head_dim == 128 && !pl->fwd_pairs && (p.flags & ARACHNE_FLAG_FWD_MULTICAST) != 0;
  // fused Q: one-CTA form, one-shard plans (tensor maps), RMSNorm on (without it the logit bound needs a pass over Q anyway)
  pl->fwd_fused_q = (p.flags & ARACHNE_FLAG_FWD_FUSED_Q) && !pl->fwd_pairs && !pl->fwd_mcast && num_shards == 1 && cp_rank < 0 &&
                    !(p.flags & ARACHNE_FLAG_NO_NORM);
  // V / dO by tensor-map TMA from the raw tensors: plain (one-shard) plans.  Token-range-sharded tensors (Ulysses, CP) have
  // tiles that straddle shards and stay on the prologue's gather; so does the CTA-pair forward (it holds half tiles).
  {
    const bool raw_ok = num_shards == 1 && !(p.flags & ARACHNE_FLAG_IMAGE_COPIES);
    pl->raw_fwd = raw_ok && !pl->fwd_pairs;
    pl->raw_bwd = raw_ok;
    pl->n_img_fwd = pl->raw_fwd ? 2 : 3;
    pl->n_img_bwd = pl->raw_bwd ? 2 : 4;
  }
  if (fwd_pair_items.empty()) fwd_pair_items.push_back(WorkItem{0, 0, 0, 0});
  pl->n_items = static_cast<int>(items.size());
  pl->n_fwd_items = static_cast<int>(fwd_items.size());
  // fwd_kernel and bwd_fused_kernel take the items of these LPT-ordered lists DYNAMICALLY (an atomic counter, sm100.cuh
  // ItemRing): list scheduling in decreasing-cost order, and CTAs that are a little faster simply take more items.
  std::vector<WorkItem> dyn_items = items, dyn_fwd_items = fwd_items;
  if (dyn_items.empty()) dyn_items.push_back(WorkItem{0, 0, 0, 0});
  if (dyn_fwd_items.empty()) dyn_fwd_items.push_back(WorkItem{0, 0, 0, 0});
  pl->n_ctas = std::min(pl->num_sms, pl->n_items);
  pl->n_fwd_ctas = std::min(pl->num_sms, pl->n_fwd_items);
  // RoPE tables in fp64 -> fp32 (readings R4, R5)
  std::vector<float2> tab;
  RopeDesc rd{};
  for (int a = 0; a < 3; ++a) {
    rd.off[a] = static_cast<int>(tab.size());
    rd.half[a] = p.rope_dims[a] / 2;
    for (int x = 0; x < ext[a]; ++x)
      for (int pr = 0; pr < rd.half[a]; ++pr) {
        const double phi = static_cast<double>(x) * std::pow(static_cast<double>(p.rope_theta), -2.0 * pr / p.rope_dims[a]);
        tab.push_back(make_float2(static_cast<float>(std::cos(phi)), static_cast<float>(std::sin(phi))));
      }
  }
  if (tab.empty()) tab.push_back(make_float2(1.f, 0.f));

  auto fail = [&](cudaError_t e, const char* what) { int rc = cuda_fail(e, what); arachne_plan_destroy(pl); return rc; };
  cudaError_t e;
#define PLAN_UP(dptr, vec, T)                                                                                   \
  if ((e = cudaMalloc(reinterpret_cast<void**>(&dptr), (vec).size() * sizeof(T))) != cudaSuccess) return fail(e, "cudaMalloc"); \
  if ((e = cudaMemcpy(dptr, (vec).data(), (vec).size() * sizeof(T), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e, "cudaMemcpy");
  PLAN_UP(pl->d_seqs, pl->seqs, SeqInfo)
  PLAN_UP(pl->d_tile_seq, tile_seq, int)
  {
    std::vector<TokInfo> ti(static_cast<size_t>(p.total_tokens));
    for (int b = 0; b < p.num_seqs; ++b) {
      const SeqInfo& s = pl->seqs[b];
      for (int n = 0; n < s.len; ++n) {
        TokInfo& x = ti[static_cast<size_t>(s.tok_start) + n];
        const bool text = n >= s.n_video;                       // R21
        const int hw = s.Hg * s.Wg;
        x.t_flag = text ? 0x80000000u : static_cast<uint32_t>(n / hw);
        x.hw = text ? 0u : (static_cast<uint32_t>((n / s.Wg) % s.Hg) << 16) | static_cast<uint32_t>(n % s.Wg);
        x.blkrow = static_cast<uint32_t>((s.tile_base + n / kTileRows) * kTileRows + n % kTileRows);
        x.seq = static_cast<uint32_t>(b);
      }
    }
    PLAN_UP(pl->d_tok_info, ti, TokInfo)
  }
  PLAN_UP(pl->d_dyn_items, dyn_items, WorkItem)
  PLAN_UP(pl->d_dyn_fwd_items, dyn_fwd_items, WorkItem)
  PLAN_UP(pl->d_dyn_fwd_pair_items, fwd_pair_items, WorkItem)
  PLAN_UP(pl->d_rope, tab, float2)
#undef PLAN_UP
  if ((e = cudaMalloc(reinterpret_cast<void**>(&pl->d_envelope), sizeof(unsigned))) != cudaSuccess) return fail(e, "cudaMalloc");
  if ((e = cudaMemset(pl->d_envelope, 0, sizeof(unsigned))) != cudaSuccess) return fail(e, "cudaMemset");
  if (pl->num_sms <= kTraceMaxCtas) {
    if ((e = cudaMalloc(reinterpret_cast<void**>(&pl->d_cta_trace), 2 * kTraceMaxCtas * 2 * sizeof(unsigned long long))) != cudaSuccess) return fail(e, "cudaMalloc");
    if ((e = cudaMemset(pl->d_cta_trace, 0, 2 * kTraceMaxCtas * 2 * sizeof(unsigned long long))) != cudaSuccess) return fail(e, "cudaMemset");
  }
  int rc = p.head_dim == 128 ? configure_kernels<128>() : configure_kernels<64>();
  if (rc != ARACHNE_OK) { arachne_plan_destroy(pl); return rc; }

  rd.tab = pl->d_rope;
  ProblemDesc& pd = pl->pd;
  pd.seqs = pl->d_seqs; pd.tile_seq = pl->d_tile_seq; pd.tok_info = pl->d_tok_info; pd.dyn_items = pl->d_dyn_items; pd.dyn_fwd_items = pl->d_dyn_fwd_items; pd.n_fwd_items = pl->n_fwd_items; pd.dyn_fwd_pair_items = pl->d_dyn_fwd_pair_items; pd.n_fwd_pair_items = pl->n_fwd_pair_items; pd.cta_trace = pl->d_cta_trace;   // stats, counters, group tables: per call (per_call_desc)
  pd.n_items = pl->n_items; pd.n_tiles_total = pl->n_tiles_total; pd.num_seqs = p.num_seqs;
  pd.N = p.total_tokens; pd.H = p.num_heads;
  pd.eps = p.rms_eps; pd.softmax_scale = pl->p.softmax_scale;
  pd.no_norm = (p.flags & ARACHNE_FLAG_NO_NORM) ? 1 : 0;
  pd.no_rope = (p.flags & ARACHNE_FLAG_NO_ROPE) ? 1 : 0;
  pd.rope = rd;
  pl->sh.n_shards = num_shards;
  for (int r = 0; r <= kMaxShards; ++r)
    pl->sh.start[r] = (shard_starts && r <= num_shards) ? shard_starts[r] : (r == 0 ? 0 : p.total_tokens);
  pl->sh.H_total = total_heads;
  pl->sh.head_offset = head_offset;
  pd.sh = pl->sh;
  {
    const long long contiguous = static_cast<long long>(total_heads) * p.head_dim;
    pd.in_stride[0] = p.q_stride ? p.q_stride : contiguous;
    pd.in_stride[1] = p.k_stride ? p.k_stride : contiguous;
    pd.in_stride[2] = p.v_stride ? p.v_stride : contiguous;
  }
  pd.cp_lo = cp_rank >= 0 ? pl->sh.start[cp_rank] : 0;
  pd.cp_hi = cp_rank >= 0 ? pl->sh.start[cp_rank + 1] : p.total_tokens;
  pl->tile_bytes = static_cast<size_t>(kTileRows) * p.head_dim * 2;
  pl->img_bytes = align_up(static_cast<size_t>(p.num_heads) * pl->n_tiles_total * pl->tile_bytes, 1024);
  pl->rowvec_bytes = align_up(static_cast<size_t>(p.num_heads) * pl->n_tiles_total * kTileRows * sizeof(float), 1024);
  pl->grad_bytes = align_up(static_cast<size_t>(p.total_tokens) * p.num_heads * p.head_dim * sizeof(float), 1024);
  pl->gradblk_bytes = align_up(static_cast<size_t>(p.num_heads) * pl->n_tiles_total * kTileRows * p.head_dim * sizeof(float), 1024);
  {
    const int tpb = 8 * (32 / (p.head_dim / 8));          // tokens per post_kernel block and step (8 warps x RPW), all heads each
    pl->post_blocks = static_cast<int>(std::min<long long>((static_cast<long long>(p.total_tokens) + tpb - 1) / tpb, static_cast<long long>(pl->num_sms) * 8));
    pl->dgpart_bytes = align_up(static_cast<size_t>(2) * pl->post_blocks * p.head_dim * sizeof(float), 1024);
  }
  pl->n_groups = p.num_seqs * p.num_heads;
  pl->hdr_bytes = align_up(sizeof(WsHeader) + static_cast<size_t>(pl->n_groups) * (16 + 16), 1024);      // header, group maxima, (sk, 1/sk, qs, 1/qs)
  {
    // Envelope (reading R19): north_star's gates are claimed for tau = softmax_scale*sqrt(D)*|gamma_q|inf*|gamma_k|inf
    // <= 1 (every BASELINE.json config has tau = 1).  The forward's logit bound in log2 units is tau*sqrt(D)*log2(e).
    const bool wide = (p.flags & (ARACHNE_FLAG_WIDE_LOGITS | ARACHNE_FLAG_NO_NORM)) != 0;
    pl->bound_limit = wide ? INFINITY : 1.001f * std::sqrt(static_cast<float>(p.head_dim)) * 1.4426950408889634f;
  }
  *out = pl;
  return ARACHNE_OK;
}
extern "C" {

void arachne_plan_destroy(arachne_plan* pl) {
  if (!pl) return;
  arachne_host_ctx_free(pl->host);
  for (auto& pass : pl->prof_ev)
    for (auto& slot : pass)
      for (cudaEvent_t ev : slot)
        if (ev) cudaEventDestroy(ev);
  cudaFree(pl->d_seqs); cudaFree(pl->d_tile_seq); cudaFree(pl->d_tok_info); cudaFree(pl->d_dyn_items); cudaFree(pl->d_dyn_fwd_items); cudaFree(pl->d_dyn_fwd_pair_items); cudaFree(pl->d_envelope); cudaFree(pl->d_cta_trace); cudaFree(pl->d_rope);
  delete pl;
}

size_t arachne_workspace_bytes(const arachne_plan* pl, int pass) {
  if (!pl) return 0;
  if (pass == 0) return fwd_ws_bytes(pl);
  if (pass == 1) return bwd_ws_bytes(pl);
  return 0;
}

int arachne_num_launches(const arachne_plan* pl, int pass) {
  if (!pl) return 0;
  if (pass == 0) return 2;                                              // prep_kernel, fwd_kernel
  if (pass == 1) return 4;                                              // prep, bwd_scale, bwd_fused, post
  return 0;
}

static int num_timed_intervals(int pass) { return pass == 0 ? 2 : (pass == 1 ? 3 : 0); }

const char* arachne_kernel_name(int pass, int idx) {
  static const char* fwd[] = {"prep_kernel(fwd: RMSNorm+RoPE -> fp16 tiles)", "fwd_kernel"};
  static const char* bwd[] = {"prep_kernel(bwd: RMSNorm+RoPE -> fp16 tiles, delta) + bwd_scale_kernel", "bwd_fused_kernel",
                              "post_kernel(un-RoPE + RMSNorm bwd)"};
  if (pass == 0 && idx >= 0 && idx < 2) return fwd[idx];
  if (pass == 1 && idx >= 0 && idx < 3) return bwd[idx];
  return "";
}

int arachne_plan_cta_times(const arachne_plan* pl, int kernel, double* start_us, double* end_us, int n, int* n_ctas) {
  if (!pl || !start_us || !end_us || !n_ctas) return ARACHNE_ERR_NULL_POINTER;
  if (kernel < 0 || kernel > 1 || !pl->d_cta_trace) return ARACHNE_ERR_BAD_PARAM;
  const int ctas = kernel == 0 ? ((pl->fwd_pairs || pl->fwd_mcast) ? pl->n_fwd_pair_ctas : pl->n_fwd_ctas) : pl->n_ctas;
  if (n < ctas) return ARACHNE_ERR_BAD_PARAM;
  std::vector<unsigned long long> t(static_cast<size_t>(kTraceMaxCtas) * 2);
  ARACHNE_CUDA(cudaMemcpy(t.data(), pl->d_cta_trace + static_cast<size_t>(kernel) * kTraceMaxCtas * 2, t.size() * sizeof(unsigned long long),
                          cudaMemcpyDeviceToHost));
  unsigned long long t0 = ~0ull;
  for (int c = 0; c < ctas; ++c) t0 = std::min(t0, t[2 * c]);
  for (int c = 0; c < ctas; ++c) { start_us[c] = (t[2 * c] - t0) * 1e-3; end_us[c] = (t[2 * c + 1] - t0) * 1e-3; }
  *n_ctas = ctas;
  return ARACHNE_OK;
}

int arachne_plan_logit_status(const arachne_plan* pl, float* tau_seen) {
  if (!pl) return ARACHNE_ERR_NULL_POINTER;
  unsigned bits = 0;
  ARACHNE_CUDA(cudaMemcpy(&bits, pl->d_envelope, sizeof(bits), cudaMemcpyDeviceToHost));
  float bound;
  std::memcpy(&bound, &bits, sizeof(bound));
  // the kernel records the logit bound in log2 units: tau * sqrt(D) * log2(e)
  const float tau = bound / (std::sqrt(static_cast<float>(pl->p.head_dim)) * 1.4426950408889634f);
  if (tau_seen) *tau_seen = bits ? tau : 0.f;
  return bits ? ARACHNE_ERR_LOGIT_RANGE : ARACHNE_OK;
}

int arachne_plan_enable_profiling(arachne_plan* pl, int enable) {
  if (!pl) return ARACHNE_ERR_NULL_POINTER;
  if (enable && !pl->prof_ev[0][0][0]) {
    for (auto& pass : pl->prof_ev)
      for (auto& slot : pass)
        for (cudaEvent_t& ev : slot) ARACHNE_CUDA(cudaEventCreate(&ev));
  }
  pl->profiling = enable != 0;
  pl->prof_calls[0] = pl->prof_calls[1] = 0;
  return ARACHNE_OK;
}

int arachne_plan_kernel_times(const arachne_plan* pl, int pass, float* ms_sum, int n_kernels, int* n_calls) {
  if (!pl || !ms_sum || !n_calls) return ARACHNE_ERR_NULL_POINTER;
  if (pass < 0 || pass > 1 || !pl->profiling) return ARACHNE_ERR_BAD_PARAM;
  const int nk = num_timed_intervals(pass);
  if (n_kernels < nk) return ARACHNE_ERR_BAD_PARAM;
  const long long calls = std::min<long long>(pl->prof_calls[pass], arachne_plan::kProfSlots);
  for (int i = 0; i < nk; ++i) ms_sum[i] = 0.f;
  for (long long c = 0; c < calls; ++c)
    for (int i = 0; i < nk; ++i) {
      float ms = 0.f;
      ARACHNE_CUDA(cudaEventSynchronize(pl->prof_ev[pass][c][i + 1]));
      ARACHNE_CUDA(cudaEventElapsedTime(&ms, pl->prof_ev[pass][c][i], pl->prof_ev[pass][c][i + 1]));
      ms_sum[i] += ms;
    }
  *n_calls = static_cast<int>(calls);
  return ARACHNE_OK;
}

namespace {
ShardedPtr one_shard(const void* p) {
  ShardedPtr s{};
  s.p[0] = const_cast<void*>(p);
  return s;
}
// copies a host array of num_shards device pointers; empty shards may be NULL; others must be 16-byte aligned
int gather_shards(const arachne_plan* pl, const void* const* arr, ShardedPtr& out) {
  out = ShardedPtr{};
  if (!arr) return ARACHNE_ERR_NULL_POINTER;
  for (int r = 0; r < pl->sh.n_shards; ++r) {
    const bool empty = pl->sh.start[r + 1] == pl->sh.start[r];
    if (!arr[r] && !empty) return ARACHNE_ERR_NULL_POINTER;
    if (misaligned(arr[r])) return ARACHNE_ERR_MISALIGNED;
    out.p[r] = const_cast<void*>(arr[r]);
  }
  return ARACHNE_OK;
}
bool row_pitch_misaligned(const arachne_plan* pl) {   // every (token, head) row must start on a 16-byte boundary
  return (static_cast<size_t>(pl->p.head_dim) * 2 * pl->sh.H_total) % 16 != 0;
}
}  // namespace

int arachne_varlen_attn_fwd(const arachne_plan* pl, const void* q, const void* k, const void* v, const float* gamma_q,
                            const float* gamma_k, void* o, float* lse, void* ws, size_t ws_bytes, void* stream) {
  if (!pl || !q || !k || !v || !o) return ARACHNE_ERR_NULL_POINTER;
  if (pl->sh.n_shards != 1) return ARACHNE_ERR_BAD_SHARDING;      // a sharded plan needs the _sharded entry points
  const void* qa[1] = {q}; const void* ka[1] = {k}; const void* va[1] = {v}; void* oa[1] = {o};
  return arachne_varlen_attn_fwd_sharded(pl, qa, ka, va, gamma_q, gamma_k, oa, lse, ws, ws_bytes, stream);
}

int arachne_varlen_attn_fwd_sharded(const arachne_plan* pl, const void* const* q, const void* const* k, const void* const* v,
                                    const float* gamma_q, const float* gamma_k, void* const* o, float* lse, void* ws,
                                    size_t ws_bytes, void* stream) {
  if (!pl || !q || !k || !v || !o || !lse || !ws) return ARACHNE_ERR_NULL_POINTER;
  ShardedPtr sq, sk, sv, so;
  int rc;
  if ((rc = gather_shards(pl, q, sq)) || (rc = gather_shards(pl, k, sk)) || (rc = gather_shards(pl, v, sv)) ||
      (rc = gather_shards(pl, o, so)))
    return rc;
  if (misaligned(lse) || misaligned(ws) || (gamma_q && misaligned(gamma_q)) || (gamma_k && misaligned(gamma_k)) ||
      row_pitch_misaligned(pl))
    return ARACHNE_ERR_MISALIGNED;
  if (ws_bytes < fwd_ws_bytes(pl)) return ARACHNE_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  return pl->p.head_dim == 128 ? launch_fwd<128>(pl, sq, sk, sv, gamma_q, gamma_k, so, lse, ws, st)
                               : launch_fwd<64>(pl, sq, sk, sv, gamma_q, gamma_k, so, lse, ws, st);
}

int arachne_varlen_attn_bwd(const arachne_plan* pl, const void* q, const void* k, const void* v, const float* gamma_q,
                            const float* gamma_k, const void* o, const float* lse, const void* d_o, void* dq, void* dk,
                            void* dv, void* ws, size_t ws_bytes, void* stream) {
  return arachne_varlen_attn_bwd_dgamma(pl, q, k, v, gamma_q, gamma_k, o, lse, d_o, dq, dk, dv, nullptr, nullptr, ws, ws_bytes, stream);
}

int arachne_varlen_attn_bwd_dgamma(const arachne_plan* pl, const void* q, const void* k, const void* v, const float* gamma_q,
                                   const float* gamma_k, const void* o, const float* lse, const void* d_o, void* dq, void* dk,
                                   void* dv, float* dgamma_q, float* dgamma_k, void* ws, size_t ws_bytes, void* stream) {
  if (!pl || !q || !k || !v || !o || !d_o || !dq || !dk || !dv) return ARACHNE_ERR_NULL_POINTER;
  if (pl->sh.n_shards != 1) return ARACHNE_ERR_BAD_SHARDING;
  const void* qa[1] = {q}; const void* ka[1] = {k}; const void* va[1] = {v}; const void* oa[1] = {o};
  const void* ga[1] = {d_o}; void* dqa[1] = {dq}; void* dka[1] = {dk}; void* dva[1] = {dv};
  return arachne_varlen_attn_bwd_sharded(pl, qa, ka, va, gamma_q, gamma_k, oa, lse, ga, dqa, dka, dva, dgamma_q, dgamma_k,
                                         ws, ws_bytes, stream);
}

int arachne_varlen_attn_bwd_sharded(const arachne_plan* pl, const void* const* q, const void* const* k, const void* const* v,
                                    const float* gamma_q, const float* gamma_k, const void* const* o, const float* lse,
                                    const void* const* d_o, void* const* dq, void* const* dk, void* const* dv,
                                    float* dgamma_q, float* dgamma_k, void* ws, size_t ws_bytes, void* stream) {
  if (!pl || !q || !k || !v || !o || !lse || !d_o || !dq || !dk || !dv || !ws) return ARACHNE_ERR_NULL_POINTER;
  if (pl->cp_rank >= 0) return ARACHNE_ERR_BAD_SHARDING;      // a context-parallel plan needs bwd_cp_partial + cp_reduce
  ShardedPtr sq, sk, sv, so, sg, sdq, sdk, sdv;
  int rc;
  if ((rc = gather_shards(pl, q, sq)) || (rc = gather_shards(pl, k, sk)) || (rc = gather_shards(pl, v, sv)) ||
      (rc = gather_shards(pl, o, so)) || (rc = gather_shards(pl, d_o, sg)) || (rc = gather_shards(pl, dq, sdq)) ||
      (rc = gather_shards(pl, dk, sdk)) || (rc = gather_shards(pl, dv, sdv)))
    return rc;
  if (misaligned(lse) || misaligned(ws) || (gamma_q && misaligned(gamma_q)) || (gamma_k && misaligned(gamma_k)) ||
      (dgamma_q && misaligned(dgamma_q)) || (dgamma_k && misaligned(dgamma_k)) || row_pitch_misaligned(pl))
    return ARACHNE_ERR_MISALIGNED;
  if (ws_bytes < bwd_ws_bytes(pl)) return ARACHNE_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  return pl->p.head_dim == 128
             ? launch_bwd<128>(pl, sq, sk, sv, gamma_q, gamma_k, so, lse, sg, sdq, sdk, sdv, dgamma_q, dgamma_k, ws, st)
             : launch_bwd<64>(pl, sq, sk, sv, gamma_q, gamma_k, so, lse, sg, sdq, sdk, sdv, dgamma_q, dgamma_k, ws, st);
}

int arachne_varlen_attn_bwd_cp_partial(const arachne_plan* pl, const void* const* q, const void* const* k,
                                       const void* const* v, const float* gamma_q, const float* gamma_k,
                                       const void* const* o, const float* lse, const void* const* d_o, void* const* dq,
                                       float* dk_partial, float* dv_partial, float* dgamma_q, void* ws, size_t ws_bytes,
                                       void* stream) {
  if (!pl || !q || !k || !v || !o || !lse || !d_o || !dq || !dk_partial || !dv_partial || !ws) return ARACHNE_ERR_NULL_POINTER;
  if (pl->cp_rank < 0) return ARACHNE_ERR_BAD_SHARDING;
  ShardedPtr sq, sk, sv, so, sg, sdq, none{};
  int rc;
  if ((rc = gather_shards(pl, q, sq)) || (rc = gather_shards(pl, k, sk)) || (rc = gather_shards(pl, v, sv)) ||
      (rc = gather_shards(pl, o, so)) || (rc = gather_shards(pl, d_o, sg)) || (rc = gather_shards(pl, dq, sdq)))
    return rc;
  if (misaligned(lse) || misaligned(ws) || misaligned(dk_partial) || misaligned(dv_partial) ||
      (gamma_q && misaligned(gamma_q)) || (gamma_k && misaligned(gamma_k)) || (dgamma_q && misaligned(dgamma_q)) ||
      row_pitch_misaligned(pl))
    return ARACHNE_ERR_MISALIGNED;
  if (ws_bytes < bwd_ws_bytes(pl)) return ARACHNE_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  return pl->p.head_dim == 128
             ? launch_bwd<128>(pl, sq, sk, sv, gamma_q, gamma_k, so, lse, sg, sdq, none, none, dgamma_q, nullptr, ws, st, dk_partial, dv_partial)
             : launch_bwd<64>(pl, sq, sk, sv, gamma_q, gamma_k, so, lse, sg, sdq, none, none, dgamma_q, nullptr, ws, st, dk_partial, dv_partial);
}

}  // extern "C"
namespace {
template <int D>
int launch_cp_reduce(const arachne_plan* pl, const ShardedPtr& gkp, const ShardedPtr& gvp, const ShardedPtr& k, const float* gk,
                     const ShardedPtr& dk, const ShardedPtr& dv, float* dgk, void* ws, cudaStream_t st) {
  uint8_t* w = static_cast<uint8_t*>(ws);
  w += pl->hdr_bytes + pl->n_img_bwd * pl->img_bytes + 3 * pl->rowvec_bytes;   // same carving as launch_bwd: gk_t, gq_t, dgamma partials
  float* gk_sum = reinterpret_cast<float*>(w); w += pl->grad_bytes + pl->gradblk_bytes;
  float* dgpart = dgk ? reinterpret_cast<float*>(w) : nullptr;
  const int lo = pl->pd.cp_lo, hi = pl->pd.cp_hi;
  if (hi > lo) {
    CpReduceParams cp{gkp, gvp, gk_sum, dv, lo, hi};
    const long long n_vec = static_cast<long long>(hi - lo) * pl->p.num_heads * (D / 4);
    const int grid = static_cast<int>(std::min<long long>((n_vec + 255) / 256, static_cast<long long>(pl->num_sms) * 8));
    cp_reduce_kernel<D><<<grid, 256, 0, st>>>(pl->pd, cp);
    ARACHNE_CUDA(cudaGetLastError());
  }
  ShardedPtr none{};
  PostParams po{nullptr, 0, 0, gk_sum, none, k, nullptr, gk, none, dk, 2, lo, hi, dgpart, nullptr};
  post_kernel<D><<<dim3(pl->post_blocks, 1), 256, 0, st>>>(pl->pd, po);
  ARACHNE_CUDA(cudaGetLastError());
  if (dgpart) {
    dgamma_reduce_kernel<D><<<2, 256, 0, st>>>(dgpart, pl->post_blocks, nullptr, dgk);
    ARACHNE_CUDA(cudaGetLastError());
  }
  return ARACHNE_OK;
}
}  // namespace
extern "C" {

int arachne_cp_reduce(const arachne_plan* pl, const float* const* dk_partials, const float* const* dv_partials,
                      const void* const* k, const float* gamma_k, void* const* dk, void* const* dv, float* dgamma_k,
                      void* ws, size_t ws_bytes, void* stream) {
  if (!pl || !dk_partials || !dv_partials || !k || !dk || !dv || !ws) return ARACHNE_ERR_NULL_POINTER;
  if (pl->cp_rank < 0) return ARACHNE_ERR_BAD_SHARDING;
  ShardedPtr gkp{}, gvp{}, sk, sdk, sdv;
  for (int r = 0; r < pl->sh.n_shards; ++r) {       // a partial buffer may be NULL only for a rank that owns no queries
    const bool empty = pl->sh.start[r + 1] == pl->sh.start[r];
    if ((!dk_partials[r] || !dv_partials[r]) && !empty) return ARACHNE_ERR_NULL_POINTER;
    if (misaligned(dk_partials[r]) || misaligned(dv_partials[r])) return ARACHNE_ERR_MISALIGNED;
    gkp.p[r] = const_cast<float*>(dk_partials[r]);
    gvp.p[r] = const_cast<float*>(dv_partials[r]);
  }
  int rc;
  if ((rc = gather_shards(pl, k, sk)) || (rc = gather_shards(pl, dk, sdk)) || (rc = gather_shards(pl, dv, sdv))) return rc;
  if (misaligned(ws) || (gamma_k && misaligned(gamma_k)) || (dgamma_k && misaligned(dgamma_k)) || row_pitch_misaligned(pl))
    return ARACHNE_ERR_MISALIGNED;
  if (ws_bytes < bwd_ws_bytes(pl)) return ARACHNE_ERR_WORKSPACE_TOO_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  return pl->p.head_dim == 128 ? launch_cp_reduce<128>(pl, gkp, gvp, sk, gamma_k, sdk, sdv, dgamma_k, ws, st)
                               : launch_cp_reduce<64>(pl, gkp, gvp, sk, gamma_k, sdk, sdv, dgamma_k, ws, st);
}

// ---------------------------------------------------------------- CUDA IPC plumbing for peer shards
int arachne_ipc_alloc(size_t bytes, void** dev_ptr, void* handle_out) {
  if (!dev_ptr || !handle_out) return ARACHNE_ERR_NULL_POINTER;
  if (bytes == 0) return ARACHNE_ERR_BAD_SHAPE;
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "handle size");
  ARACHNE_CUDA(cudaMalloc(dev_ptr, bytes));
  cudaIpcMemHandle_t h;
  cudaError_t e = cudaIpcGetMemHandle(&h, *dev_ptr);
  if (e != cudaSuccess) { cudaFree(*dev_ptr); *dev_ptr = nullptr; return cuda_fail(e, "cudaIpcGetMemHandle"); }
  std::memcpy(handle_out, &h, sizeof(h));
  return ARACHNE_OK;
}
int arachne_ipc_open(const void* handle, void** dev_ptr) {
  if (!handle || !dev_ptr) return ARACHNE_ERR_NULL_POINTER;
  cudaIpcMemHandle_t h;
  std::memcpy(&h, handle, sizeof(h));
  ARACHNE_CUDA(cudaIpcOpenMemHandle(dev_ptr, h, cudaIpcMemLazyEnablePeerAccess));
  return ARACHNE_OK;
}
int arachne_ipc_close(void* dev_ptr) {
  if (!dev_ptr) return ARACHNE_ERR_NULL_POINTER;
  ARACHNE_CUDA(cudaIpcCloseMemHandle(dev_ptr));
  return ARACHNE_OK;
}
int arachne_ipc_free(void* dev_ptr) {
  if (!dev_ptr) return ARACHNE_ERR_NULL_POINTER;
  ARACHNE_CUDA(cudaFree(dev_ptr));
  return ARACHNE_OK;
}

// ---------------------------------------------------------------- host-buffer convenience calls
// Device buffers and the two streams are created on the first host call and cached in the plan (freed by
// arachne_plan_destroy).  Copies overlap the kernels: dO goes up while the forward runs, O and LSE come down while
// the backward runs; PCIe is full duplex, so only Q,K,V in front and dQ,dK,dV at the end are exposed.
struct arachne_host_ctx {
  void *q = nullptr, *k = nullptr, *v = nullptr, *o = nullptr, *lse = nullptr, *ws = nullptr, *d_o = nullptr, *dq = nullptr,
       *dk = nullptr, *dv = nullptr, *gq = nullptr, *gk = nullptr;
  size_t ws_bytes = 0;
  bool has_bwd = false;
  cudaStream_t compute = nullptr, copy = nullptr;
  cudaEvent_t ev_do_up = nullptr, ev_fwd = nullptr, ev_o_down = nullptr, ev_dv = nullptr;
  ~arachne_host_ctx() {
    for (void* p : {q, k, v, o, lse, ws, d_o, dq, dk, dv, gq, gk}) cudaFree(p);
    for (cudaEvent_t e : {ev_do_up, ev_fwd, ev_o_down, ev_dv}) if (e) cudaEventDestroy(e);
    if (compute) cudaStreamDestroy(compute);
    if (copy) cudaStreamDestroy(copy);
  }
};

}  // extern "C"
static void arachne_host_ctx_free(arachne_host_ctx* c) { delete c; }
extern "C" {

static int host_ctx_fill(const arachne_plan* pl, bool with_bwd, arachne_host_ctx* c, bool fresh) {
  const size_t nb = static_cast<size_t>(pl->p.total_tokens) * pl->p.num_heads * pl->p.head_dim * 2;
  const size_t lb = static_cast<size_t>(pl->p.total_tokens) * pl->p.num_heads * sizeof(float);
  const size_t gb = static_cast<size_t>(pl->p.head_dim) * sizeof(float);
  if (fresh) {
    ARACHNE_CUDA(cudaStreamCreateWithFlags(&c->compute, cudaStreamNonBlocking));
    ARACHNE_CUDA(cudaStreamCreateWithFlags(&c->copy, cudaStreamNonBlocking));
    for (cudaEvent_t* e : {&c->ev_do_up, &c->ev_fwd, &c->ev_o_down, &c->ev_dv})
      ARACHNE_CUDA(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    ARACHNE_CUDA(cudaMalloc(&c->q, nb)); ARACHNE_CUDA(cudaMalloc(&c->k, nb)); ARACHNE_CUDA(cudaMalloc(&c->v, nb));
    ARACHNE_CUDA(cudaMalloc(&c->o, nb)); ARACHNE_CUDA(cudaMalloc(&c->lse, lb));
    ARACHNE_CUDA(cudaMalloc(&c->gq, gb)); ARACHNE_CUDA(cudaMalloc(&c->gk, gb));
  }
  const size_t wsb = std::max(fwd_ws_bytes(pl), with_bwd ? bwd_ws_bytes(pl) : size_t(0));
  if (c->ws_bytes < wsb) {
    ARACHNE_CUDA(cudaFree(c->ws)); c->ws = nullptr; c->ws_bytes = 0;
    ARACHNE_CUDA(cudaMalloc(&c->ws, wsb)); c->ws_bytes = wsb;
  }
  if (with_bwd && !c->has_bwd) {
    ARACHNE_CUDA(cudaMalloc(&c->d_o, nb)); ARACHNE_CUDA(cudaMalloc(&c->dq, nb));
    ARACHNE_CUDA(cudaMalloc(&c->dk, nb)); ARACHNE_CUDA(cudaMalloc(&c->dv, nb));
    c->has_bwd = true;
  }
  return ARACHNE_OK;
}

// The context is cached in the plan only once EVERY allocation has succeeded: a failed cudaMalloc (e.g. out of memory on a
// 262K-token batch) frees whatever was built and leaves the plan as it was, so the next host call starts from scratch
// instead of running on null buffers.
static int host_ctx(const arachne_plan* pl, bool with_bwd, arachne_host_ctx** out) {
  arachne_host_ctx* c = pl->host;
  const bool fresh = c == nullptr;
  if (fresh) {
    c = new (std::nothrow) arachne_host_ctx();
    if (!c) { g_last_error = "out of host memory"; return ARACHNE_ERR_CUDA; }
  }
  const int rc = host_ctx_fill(pl, with_bwd, c, fresh);
  if (rc != ARACHNE_OK) {
    if (!fresh) pl->host = nullptr;
    delete c;                        // frees every buffer, event and stream it holds
    return rc;
  }
  pl->host = c;
  *out = c;
  return ARACHNE_OK;
}

static int run_host_enqueue(const arachne_plan* pl, arachne_host_ctx* c, bool with_bwd, const void* q_h, const void* k_h,
                            const void* v_h, const float* gq_h, const float* gk_h, const void* do_h, void* o_h, float* lse_h,
                            void* dq_h, void* dk_h, void* dv_h);

static int run_host(const arachne_plan* pl, bool with_bwd, const void* q_h, const void* k_h, const void* v_h,
                    const float* gq_h, const float* gk_h, const void* do_h, void* o_h, float* lse_h, void* dq_h,
                    void* dk_h, void* dv_h) {
  if (!pl || !q_h || !k_h || !v_h || !o_h || !lse_h) return ARACHNE_ERR_NULL_POINTER;
  if (with_bwd && (!do_h || !dq_h || !dk_h || !dv_h)) return ARACHNE_ERR_NULL_POINTER;
  if (pl->sh.n_shards != 1) return ARACHNE_ERR_BAD_SHARDING;
  if (pl->p.q_stride || pl->p.k_stride || pl->p.v_stride) return ARACHNE_ERR_BAD_PARAM;     // host buffers are dense [N, H, D]
  arachne_host_ctx* c = nullptr;
  int rc = host_ctx(pl, with_bwd, &c);
  if (rc) return rc;
  rc = run_host_enqueue(pl, c, with_bwd, q_h, k_h, v_h, gq_h, gk_h, do_h, o_h, lse_h, dq_h, dk_h, dv_h);
  // whatever happened, nothing is left running on the private streams when the call returns
  const cudaError_t e1 = cudaStreamSynchronize(c->copy), e2 = cudaStreamSynchronize(c->compute);
  if (rc == ARACHNE_OK && e1 != cudaSuccess) return cuda_fail(e1, "cudaStreamSynchronize(copy)");
  if (rc == ARACHNE_OK && e2 != cudaSuccess) return cuda_fail(e2, "cudaStreamSynchronize(compute)");
  return rc;
}

static int run_host_enqueue(const arachne_plan* pl, arachne_host_ctx* c, bool with_bwd, const void* q_h, const void* k_h,
                            const void* v_h, const float* gq_h, const float* gk_h, const void* do_h, void* o_h, float* lse_h,
                            void* dq_h, void* dk_h, void* dv_h) {
  const size_t nb = static_cast<size_t>(pl->p.total_tokens) * pl->p.num_heads * pl->p.head_dim * 2;
  const size_t lb = static_cast<size_t>(pl->p.total_tokens) * pl->p.num_heads * sizeof(float);
  const size_t gb = static_cast<size_t>(pl->p.head_dim) * sizeof(float);
  int rc;
  cudaStream_t st = c->compute, cp = c->copy;
  float* gq = gq_h ? static_cast<float*>(c->gq) : nullptr;
  float* gk = gk_h ? static_cast<float*>(c->gk) : nullptr;
  ARACHNE_CUDA(cudaMemcpyAsync(c->q, q_h, nb, cudaMemcpyHostToDevice, st));
  ARACHNE_CUDA(cudaMemcpyAsync(c->k, k_h, nb, cudaMemcpyHostToDevice, st));
  ARACHNE_CUDA(cudaMemcpyAsync(c->v, v_h, nb, cudaMemcpyHostToDevice, st));
  if (gq) ARACHNE_CUDA(cudaMemcpyAsync(gq, gq_h, gb, cudaMemcpyHostToDevice, st));
  if (gk) ARACHNE_CUDA(cudaMemcpyAsync(gk, gk_h, gb, cudaMemcpyHostToDevice, st));
  if (with_bwd) {      // dO rides up behind Q,K,V on the copy stream while the forward kernels run
    ARACHNE_CUDA(cudaEventRecord(c->ev_fwd, st));               // (here: Q,K,V copies issued; keeps the link in order)
    ARACHNE_CUDA(cudaStreamWaitEvent(cp, c->ev_fwd, 0));
    ARACHNE_CUDA(cudaMemcpyAsync(c->d_o, do_h, nb, cudaMemcpyHostToDevice, cp));
    ARACHNE_CUDA(cudaEventRecord(c->ev_do_up, cp));
  }
  rc = arachne_varlen_attn_fwd(pl, c->q, c->k, c->v, gq, gk, c->o, static_cast<float*>(c->lse), c->ws, c->ws_bytes, st);
  if (rc) return rc;
  ARACHNE_CUDA(cudaEventRecord(c->ev_fwd, st));
  // O and LSE come down on the copy stream while the backward runs
  ARACHNE_CUDA(cudaStreamWaitEvent(cp, c->ev_fwd, 0));
  ARACHNE_CUDA(cudaMemcpyAsync(o_h, c->o, nb, cudaMemcpyDeviceToHost, cp));
  ARACHNE_CUDA(cudaMemcpyAsync(lse_h, c->lse, lb, cudaMemcpyDeviceToHost, cp));
  ARACHNE_CUDA(cudaEventRecord(c->ev_o_down, cp));
  if (with_bwd) {
    ARACHNE_CUDA(cudaStreamWaitEvent(st, c->ev_do_up, 0));
    rc = arachne_varlen_attn_bwd(pl, c->q, c->k, c->v, gq, gk, c->o, static_cast<float*>(c->lse), c->d_o, c->dq, c->dk,
                                 c->dv, c->ws, c->ws_bytes, st);
    if (rc) return rc;
    ARACHNE_CUDA(cudaMemcpyAsync(dv_h, c->dv, nb, cudaMemcpyDeviceToHost, st));
    ARACHNE_CUDA(cudaMemcpyAsync(dq_h, c->dq, nb, cudaMemcpyDeviceToHost, st));
    ARACHNE_CUDA(cudaMemcpyAsync(dk_h, c->dk, nb, cudaMemcpyDeviceToHost, st));
  }
  return ARACHNE_OK;
}

int arachne_varlen_attn_fwd_host(const arachne_plan* pl, const void* q_h, const void* k_h, const void* v_h,
                                 const float* gq_h, const float* gk_h, void* o_h, float* lse_h) {
  return run_host(pl, false, q_h, k_h, v_h, gq_h, gk_h, nullptr, o_h, lse_h, nullptr, nullptr, nullptr);
}

int arachne_varlen_attn_fwd_bwd_host(const arachne_plan* pl, const void* q_h, const void* k_h, const void* v_h,
                                     const float* gq_h, const float* gk_h, const void* do_h, void* o_h, float* lse_h,
                                     void* dq_h, void* dk_h, void* dv_h) {
  return run_host(pl, true, q_h, k_h, v_h, gq_h, gk_h, do_h, o_h, lse_h, dq_h, dk_h, dv_h);
}

}  // extern "C"

// ---------------------------------------------------------------- forward without any caller- or library-allocated scratch
// arachne_varlen_attn_fwd_noalloc (include/arachne_attn.h): for callers that cannot get device memory at all — a layer
// living inside a process whose framework allocator already holds the GPU's memory, a C host that only ever receives
// tensor pointers from its embedder, a step loop in which cudaMalloc / cudaFree are forbidden because they stall the
// device.  The forward's scratch (workspace header + Q^ / K^ operand images) is this array instead of a workspace argument.
//
// The array is part of the library's device image: every GPU that loads the image holds kBuiltinScratchBytes of it until the
// process ends.  In HOST code the identifier below is only a handle for the runtime's symbol table, never a device address
// (handing it to a kernel would fault, or quietly address host memory where the GPU can reach it): the host side must ask
// cudaGetSymbolAddress, with the right device current, and pass the pointer it gets.  Kernels in this file could also name
// the array directly; launch_fwd's kernels take the workspace as a pointer, so the pointer route serves both entry points.
constexpr size_t kBuiltinScratchBytes = ARACHNE_BUILTIN_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_builtin_scratch[kBuiltinScratchBytes];

namespace {
constexpr int kMaxBuiltinDevices = 64;
std::mutex g_builtin_mu;
void* g_builtin_ptr[kMaxBuiltinDevices] = {};      // device address of g_builtin_scratch on device i (0 = not looked up yet)

// Once per device, with that device current.  Not an allocation — the bytes came with the module — but the look-up may be
// what makes a lazily-loading runtime bring the module in, hence the header's "first call before any stream capture".
int builtin_scratch(int dev, void** out) {
  if (dev < 0 || dev >= kMaxBuiltinDevices) { g_last_error = "device ordinal beyond the built-in scratch table"; return ARACHNE_ERR_BAD_PARAM; }
  std::lock_guard<std::mutex> lock(g_builtin_mu);
  if (!g_builtin_ptr[dev]) {
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_builtin_scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_builtin_scratch)");
    if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) { g_last_error = "built-in scratch: bad symbol address"; return ARACHNE_ERR_CUDA; }
    g_builtin_ptr[dev] = ptr;
  }
  *out = g_builtin_ptr[dev];
  return ARACHNE_OK;
}
}  // namespace

extern "C" int arachne_varlen_attn_fwd_noalloc(const arachne_plan* pl, const void* q, const void* k, const void* v,
                                               const float* gamma_q, const float* gamma_k, void* o, float* lse,
                                               void* stream) {
  if (!pl || !q || !k || !v || !o || !lse) return ARACHNE_ERR_NULL_POINTER;
  if (pl->sh.n_shards != 1) return ARACHNE_ERR_BAD_SHARDING;
  const size_t need = fwd_ws_bytes(pl);
  if (need > kBuiltinScratchBytes) {      // refused before anything is enqueued
    g_last_error = "arachne_varlen_attn_fwd_noalloc: this packing needs " + std::to_string(need) + " bytes of scratch, the built-in array has " +
                   std::to_string(kBuiltinScratchBytes) + "; call arachne_varlen_attn_fwd with a workspace instead";
    return ARACHNE_ERR_BUILTIN_SCRATCH;
  }
  int dev = -1;
  ARACHNE_CUDA(cudaGetDevice(&dev));
  if (dev != pl->device) { g_last_error = "arachne_varlen_attn_fwd_noalloc: the plan was built on another device than the current one"; return ARACHNE_ERR_BAD_PARAM; }
  void* scratch = nullptr;
  const int rc = builtin_scratch(dev, &scratch);
  if (rc != ARACHNE_OK) return rc;
  // From here on this IS arachne_varlen_attn_fwd: same validation, same launches (launch_fwd clears the workspace header —
  // the only words that must start at zero — on the stream before the prologue; the operand images, tail padding
  // included, are written by the prologue before fwd_kernel reads them), with the built-in array as the workspace.
  return arachne_varlen_attn_fwd(pl, q, k, v, gamma_q, gamma_k, o, lse, scratch, kBuiltinScratchBytes, stream);
}
