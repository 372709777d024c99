/* arachne_attn.h — C ABI of libarachne_attn.so (B200 / sm_100a only).
 *
 * One operation: a DiT block's full 3D self-attention, forward and backward, over a PACKED
 * batch of heterogeneous-length video-latent token sequences (block-diagonal: a token
 * attends only to tokens of its own sequence), with QK-RMSNorm and 3D (t,h,w) RoPE applied
 * to Q and K on the way in.
 *
 * Where the operation is defined.  The paper (Arachne, arxiv 2607.01701; PAPER.md) only
 * NAMES it: "the DiT architecture's full self-attention over a unified sequence of 3D
 * patches of length L, which incurs quadratic (O(L^2)) complexity ... the dominant
 * performance bottleneck" (§III Observation 2; the alpha2*B*S^2 term of
 * Eq. 9).  It gives no formula for the attention itself.  The exact
 * arithmetic is therefore fixed by BASELINE.json (north_star, configs[0]) and the readings
 * R1-R18 listed in DESIGN.md §3; the defining equations are restated in DESIGN.md §2 and
 * implemented, independently of this library, by oracle/arachne_oracle.c.
 *
 *   x^      = gamma * x / sqrt(mean_d(x_d^2) + eps)          (per token, per head; x = Q or K row)
 *   x~      = RoPE3D(x^ ; pos(n))     pos(n) = (n / (Hg*Wg), (n / Wg) % Hg, n % Wg)
 *   s_ij    = softmax_scale * <q~_i, k~_j>                    i, j in the same sequence
 *   LSE_i   = ln sum_j exp(s_ij)      P_ij = exp(s_ij - LSE_i)      O_i = sum_j P_ij V_j
 *   backward: given dO, gradients dQ, dK (w.r.t. the RAW Q, K, through RoPE and RMSNorm) and dV.
 *
 * Conventions common to every entry point
 *   - All tensor pointers are DEVICE pointers unless the name ends in _host.
 *   - q, k, v, o, d_o, dq, dk, dv : bf16, logical shape [N, H, D], contiguous (token-major;
 *     element (n,h,d) at ((n*H)+h)*D+d).  N = total_tokens, H = num_heads, D = head_dim.
 *   - lse : fp32 [H, N] (natural log).  gamma_q, gamma_k : fp32 [D] or NULL (= all ones).
 *   - Pointers must be 16-byte aligned.  The caller owns every tensor and the workspace;
 *     the library owns only the plan.  Nothing is allocated, freed or synchronised inside
 *     fwd/bwd; all work is enqueued on `cuda_stream` (a cudaStream_t passed as void*).
 *   - Outputs are fully overwritten.  Rows of other sequences are never read or written
 *     on behalf of a sequence (block-diagonal), including at ragged tile tails.
 *   - Every function returns an arachne_status (0 = OK) and never throws or aborts.
 *     Invalid arguments are rejected before any kernel is launched.
 */
#ifndef ARACHNE_ATTN_H_
#define ARACHNE_ATTN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  ARACHNE_OK = 0,
  ARACHNE_ERR_NULL_POINTER = 1,
  ARACHNE_ERR_BAD_HEAD_DIM = 2,      /* head_dim not in {64, 128}                          */
  ARACHNE_ERR_BAD_ROPE_DIMS = 3,     /* a rope dim is odd / negative, or they do not sum to D */
  ARACHNE_ERR_BAD_CU_SEQLENS = 4,    /* cu_seqlens[0] != 0 or not strictly increasing       */
  ARACHNE_ERR_GRID_MISMATCH = 5,     /* T*Hg*Wg != cu_seqlens[b+1]-cu_seqlens[b]            */
  ARACHNE_ERR_TOTAL_TOKENS = 6,      /* cu_seqlens[B] != total_tokens                       */
  ARACHNE_ERR_MISALIGNED = 7,        /* a tensor / workspace pointer is not 16-byte aligned */
  ARACHNE_ERR_WORKSPACE_TOO_SMALL = 8,
  ARACHNE_ERR_BAD_ARCH = 9,          /* current device is not compute capability 10.x       */
  ARACHNE_ERR_CUDA = 10,             /* CUDA runtime error; text in arachne_last_error_message */
  ARACHNE_ERR_BAD_SHAPE = 11,        /* num_seqs/num_heads/total_tokens <= 0, or too large  */
  ARACHNE_ERR_BAD_PARAM = 12,        /* non-finite / non-positive theta, eps < 0, bad flags */
  ARACHNE_ERR_BAD_SHARDING = 13,     /* see arachne_plan_create_sharded; or a sharded plan passed to a plain call */
  ARACHNE_ERR_LOGIT_RANGE = 14,      /* tau > 1 without ARACHNE_FLAG_WIDE_LOGITS: see "Verified envelope" below      */
  ARACHNE_ERR_BUILTIN_SCRATCH = 15   /* arachne_varlen_attn_fwd_noalloc: the packing needs more scratch than the library's
                                        built-in ARACHNE_BUILTIN_SCRATCH_BYTES; sizes in arachne_last_error_message      */
} arachne_status;

enum {
  ARACHNE_FLAG_DETERMINISTIC = 1,    /* bwd: bit-reproducible run to run (same device, plan) */
  ARACHNE_FLAG_NO_NORM = 2,          /* debug: skip RMSNorm (x^ = x)                         */
  ARACHNE_FLAG_NO_ROPE = 4,          /* debug: skip RoPE (x~ = x^)                           */
  ARACHNE_FLAG_WIDE_LOGITS = 8,      /* the caller accepts logits outside the verified envelope (below) */
  ARACHNE_FLAG_FWD_CTA_PAIRS = 16,   /* A-B: run the forward as CTA pairs (cluster of 2, tcgen05 cta_group::2; head_dim 128
                                        only, ignored otherwise).  Correct (same parity tests) but SLOWER than the default
                                        one-CTA kernel — 720p forward 202 vs 147 ms (profiles/r2_bench_final.md): the forward loop is bound by the
                                        softmax <-> MMA hand-off latency, which the cross-CTA hops lengthen, not by the
                                        shared-memory operand bandwidth the pairing relieves           */
  ARACHNE_FLAG_FWD_MULTICAST = 64,   /* forward as clusters of 2 CTAs that share the K^/V stream: each CTA fetches half of
                                        every tile and the TMA engine multicasts it into both (head_dim 128 only, ignored
                                        otherwise); halves the L2 -> SM traffic of the forward         */
  ARACHNE_FLAG_FWD_FUSED_Q = 128,    /* A-B of SURVEY §7.2 "measure both": the forward loads its RAW query tiles and applies
                                        RMSNorm + RoPE + scale to them inside fwd_kernel (once per work item) instead of
                                        reading Q^ tile images written by the in-call prologue; same bytes reach the
                                        tensor core.  One-CTA form, one-shard plans, RMSNorm on; ignored otherwise.
                                        Slower on short sequences                                        */
  ARACHNE_FLAG_IMAGE_COPIES = 32     /* A-B: the prologue copies V (and dO) into tile images in the workspace, as round 1
                                        did, instead of the main kernels reading them from the caller's tensors by
                                        tensor-map TMA (the default for one-shard plans).  Same results
                                        bit for bit; more HBM traffic and a larger workspace                          */
};

/* Verified envelope (reading R19).  Q^ and K^ enter the tensor cores as fp16 — the most precise 16-bit
 * operand format, legal because RMSNorm bounds |x^_d| <= |gamma|inf * sqrt(D) — in the forward and, bit for bit the
 * same images, in the backward's recompute of S.  The rounding error of a logit is proportional to its size:
 * |delta s_ij| <= 2^-10 * beta with beta = softmax_scale * D * |gamma_q|inf * |gamma_k|inf the logit bound, and LSE
 * inherits it without averaging once the softmax is peaked.  Let
 *     tau = softmax_scale * sqrt(D) * |gamma_q|inf * |gamma_k|inf        (= 1 for every BASELINE.json config).
 * BASELINE.json's tolerances (O rel-L2 <= 1e-2, max-abs <= 2e-2, LSE max-abs <= 1e-3, dQ/dK/dV rel-L2 <= 2e-2) are
 * claimed for tau <= 1.  For tau > 1 the O and gradient tolerances still hold as far as they have been measured
 * (tau = 9: gamma_q = gamma_k = 3, tests/test_gpu_parity.py), but LSE is only bounded by 2^-10 * beta (measured
 * max-abs: 5e-4..1.2e-3 at tau = 1.6, 3e-3 at tau = 4, 9e-3 at tau = 9).  Because this is a precision limit and not a
 * failure, it is reported instead of hidden:
 *   - arachne_plan_create* returns ARACHNE_ERR_LOGIT_RANGE when softmax_scale * sqrt(D) > 1 (known on the host) unless
 *     ARACHNE_FLAG_WIDE_LOGITS (or the debug flag NO_NORM, whose logits are unbounded anyway) is set;
 *   - gamma lives in device memory, so |gamma|inf is only known to the kernels: a forward launched WITHOUT the flag whose
 *     tau exceeds 1 still runs, and leaves a sticky mark in the plan that arachne_plan_logit_status returns.
 * Callers with learned QK-norm weights either set the flag (accepting the LSE bound above) or poll the status. */

/* ABI version.  arachne_attn_params is passed by pointer and has grown between versions (version 2 appended q_stride, k_stride,
 * v_stride), so a caller compiled against an older header would hand the library a struct that is too short.  A caller that
 * may meet a library built from a different header checks, once, that arachne_abi_version() == ARACHNE_ABI_VERSION (the
 * value it was compiled with) and that arachne_attn_params_size() == sizeof(arachne_attn_params); binding.py does both when
 * it is imported and refuses to load otherwise.  The number changes whenever a struct layout, an enum value or the meaning
 * or argument list of an existing entry point changes; new entry points alone do not change it.
 *   1: round 1.   2: q/k/v_stride appended to arachne_attn_params.   3: arachne_workspace_bytes(plan, 1) larger (per-row
 *   fixed-point scales), status 15, this pair of functions. */
#define ARACHNE_ABI_VERSION 3
int arachne_abi_version(void);
size_t arachne_attn_params_size(void);

/* Problem description.  Plain data, copied by arachne_plan_create. */
typedef struct {
  int32_t num_seqs;       /* B                                                            */
  int32_t total_tokens;   /* N = sum_b L_b                                                */
  int32_t num_heads;      /* H                                                            */
  int32_t head_dim;       /* D in {64, 128}                                               */
  int32_t rope_dims[3];   /* (d_t, d_h, d_w): each even and >= 0, sum == head_dim; axis a
                             owns the contiguous slice of head_dim of width d_a, in this
                             order; inside a slice, pair p is elements (2p, 2p+1)          */
  float rope_theta;       /* angle = pos_a * theta^(-2p/d_a); 10000                        */
  float rms_eps;          /* added to the mean square, inside the sqrt; 1e-6               */
  float softmax_scale;    /* 0 => 1/sqrt(head_dim)                                         */
  int32_t flags;          /* ARACHNE_FLAG_*                                                */
  int64_t q_stride;       /* elements between consecutive TOKENS of Q / K / V; 0 => num_heads * head_dim   */
  int64_t k_stride;       /* (contiguous).  The heads of a token stay adjacent (head stride = head_dim),    */
  int64_t v_stride;       /* which covers the strided producers there are: a fused QKV projection           */
                          /* [N, 3, H, D] is three base pointers with stride 3*H*D.  Each must be a         */
                          /* multiple of 8 and >= num_heads * head_dim; one-shard plans only (sharded       */
                          /* plans: 0).  O, LSE, dO and the gradients are always contiguous.                */
} arachne_attn_params;

/* Q, K, V may be token-strided views (q_stride, k_stride, v_stride above): Q and K rows are read once by the
 * in-call prologue and once by the backward epilogue, V tiles by tensor-map TMA whose token stride is simply the map's.
 * Everything the library writes (O, LSE, dQ, dK, dV) and dO are contiguous [N, H, D]; the sharded entry points below cover
 * the other strided layout the method needs (a head range of a wider [n, total_heads, D] tensor). */

typedef struct arachne_plan arachne_plan;

/* A plan is IMMUTABLE schedule data (work lists, token tables, RoPE tables) plus three pieces of mutable state that the
 * hot path touches: (1) the sticky envelope word written by out-of-envelope forwards (arachne_plan_logit_status), (2) the
 * per-CTA trace of the last launch (arachne_plan_cta_times) and (3), only while arachne_plan_enable_profiling is on, the
 * timing events.  Everything a launch needs to mutate (dynamic work counters, logit bound, dS scaling tables) lives in the
 * header of the CALLER'S workspace, so one plan may serve concurrent calls on different streams provided each call has
 * its own workspace (and profiling is off); the *_host calls keep per-plan device buffers and are not re-entrant. */

/* Build the reusable schedule for one packing (a DiT cascade runs ~60 layers x
 * (2 fwd + 1 bwd) on the same packing).  Validates everything,
 * builds the tile work lists in longest-processing-time-first order (heaviest
 * (sequence, head) groups first, tiles of one group adjacent for L2 reuse of its K/V)
 * and the RoPE cos/sin tables, and uploads them to the current device.
 *   cu_seqlens_host : int32 [B+1] HOST, cu_seqlens[0] = 0, strictly increasing, [B] = N
 *   grids_host      : int32 [B][3] HOST = (T, Hg, Wg) latent grid of each sequence;
 *                     tokens of a sequence are in row-major (t, h, w) order, w fastest
 * On success *out owns host + small device arrays; free with arachne_plan_destroy.
 * Synchronous (uses cudaMalloc/cudaMemcpy). */
int arachne_plan_create(arachne_plan** out, const arachne_attn_params* params,
                        const int32_t* cu_seqlens_host, const int32_t* grids_host);
/* Same, for JOINT sequences (the single-stream blocks of HunyuanVideo and CogVideoX's
 * full attention run over video and text tokens together; text "< 256 tokens", PAPER.md:201;
 * DESIGN.md reading R21): sequence b = its T*Hg*Wg video tokens in row-major (t,h,w) order FOLLOWED by
 * text_lens_host[b] >= 0 text tokens, cu_seqlens[b+1]-cu_seqlens[b] == T*Hg*Wg + text_lens_host[b].  Text
 * tokens get the same QK-RMSNorm but NO RoPE; attention is full over all tokens of the sequence.
 *   text_lens_host : int32 [B] HOST, or NULL (= all zero, identical to arachne_plan_create)
 * Errors: a negative text length is ARACHNE_ERR_BAD_SHAPE; a length mismatch ARACHNE_ERR_GRID_MISMATCH. */
int arachne_plan_create_joint(arachne_plan** out, const arachne_attn_params* params,
                              const int32_t* cu_seqlens_host, const int32_t* grids_host,
                              const int32_t* text_lens_host);
/* Plan for Ulysses sequence parallelism with the All-to-All FUSED into the kernels (
 * PAPER.md:84 "Ulysses SP partitions along the attention-head dimension ... All-to-All"; the SP degree k is what
 * Arachne tunes per cascade).  The packed batch of N tokens is split BY TOKEN RANGE into
 * num_shards buffers (one per SP rank): shard r is a [n_r, total_heads, D] bf16 tensor holding the global tokens
 * [shard_starts_host[r], shard_starts_host[r+1]) with ALL heads — exactly what rank r has before Ulysses'
 * first All-to-All.  This process computes heads [head_offset, head_offset + params->num_heads) of EVERY
 * token: the *_sharded calls read Q, K, V (and O, dO) rows of those heads straight out of all shards and write
 * O (dQ, dK, dV) rows of those heads straight into them.  A shard pointer may be local memory or a peer GPU's
 * memory mapped into this process (CUDA IPC / symmetric memory over NVLink-NVSwitch): the gather IS the first
 * All-to-All and the scatter IS the second, with no staging buffer, overlapped with the tensor-core kernels.
 * The caller orders the ranks (all shards written before any rank's call starts; all calls finished before a
 * shard is read): paper_2607_01701_b200/ulysses.py does it with torch.distributed barriers.
 *   params->num_heads : LOCAL head count;  total_heads : heads in the raw tensors;  cu_seqlens / grids / text_lens
 *   describe the GLOBAL pack (sequences may straddle shard boundaries);  1 <= num_shards <= 8;  shard_starts_host
 *   int32 [num_shards+1] HOST, [0] = 0, non-decreasing, [num_shards] = N (NULL allowed iff num_shards == 1).
 * lse, the workspace, gamma and dgamma are LOCAL: lse fp32 [num_heads, N]; dgamma is this rank's partial sum over
 * its heads (all-reduce it across the SP group).  Errors: ARACHNE_ERR_BAD_SHARDING. */
int arachne_plan_create_sharded(arachne_plan** out, const arachne_attn_params* params,
                                const int32_t* cu_seqlens_host, const int32_t* grids_host,
                                const int32_t* text_lens_host, int32_t num_shards,
                                const int32_t* shard_starts_host, int32_t total_heads, int32_t head_offset);
void arachne_plan_destroy(arachne_plan* plan);

/* Bytes of caller-owned device workspace needed by one call.  pass: 0 = fwd, 1 = bwd.
 * Returns 0 if plan is NULL or pass is invalid. */
size_t arachne_workspace_bytes(const arachne_plan* plan, int pass);

/* Number of kernels one arachne_varlen_attn_fwd (pass 0) / arachne_varlen_attn_bwd (pass 1) call enqueues, for launch
 * accounting: fwd 2 (prep, fwd); bwd 4 (prep, bwd_scale, bwd_fused, post); the _dgamma form adds one. */
int arachne_num_launches(const arachne_plan* plan, int pass);

/* Name of TIMED INTERVAL `idx` (0-based, launch order) of a pass — the unit arachne_plan_kernel_times reports: fwd has 2
 * (prep_kernel, fwd_kernel), bwd has 3 (prep + bwd_scale, bwd_fused_kernel, post [+ dgamma reduce]); "" if out of range. */
const char* arachne_kernel_name(int pass, int idx);

/* Sticky envelope status of a plan ("Verified envelope" above).  ARACHNE_OK if no forward launched on this plan without
 * ARACHNE_FLAG_WIDE_LOGITS has seen tau > 1; else ARACHNE_ERR_LOGIT_RANGE and *tau_seen (nullable) = the largest tau.
 * Synchronous (cudaMemcpy of 4 bytes): call it after the stream has been synchronised. */
int arachne_plan_logit_status(const arachne_plan* plan, float* tau_seen);

/* Per-kernel device timing for benchmarks (bench.py's roofline figure).  When enabled, fwd/bwd
 * record a CUDA event before the first and after every kernel on the caller's stream (no
 * synchronisation is added); the plan keeps the events of the last 32 calls per pass.
 * arachne_plan_kernel_times synchronises on those events and writes to ms_sum[i] the SUM over
 * the recorded calls of timed interval i's duration in milliseconds (ms_sum has n_kernels >= 2 (fwd) / 3 (bwd)
 * entries, see arachne_kernel_name) and the number of calls to *n_calls.  Enabling resets the ring.
 * Not thread-safe with concurrent fwd/bwd on the same plan. */
int arachne_plan_enable_profiling(arachne_plan* plan, int enable);
int arachne_plan_kernel_times(const arachne_plan* plan, int pass, float* ms_sum, int n_kernels, int* n_calls);

/* Per-CTA trace of the LAST launch of a persistent kernel (kernel: 0 = fwd_kernel, 1 = bwd_fused_kernel): every CTA
 * stamps %globaltimer when it starts and when it has finished its last work item (two 8-byte stores per CTA; always on).
 * Writes start_us[c], end_us[c] (microseconds since the earliest CTA start) for c < *n_ctas; n = capacity of the arrays
 * (>= the SM count).  Synchronous (cudaMemcpy): call it after the stream has been synchronised.  The spread of end_us is
 * the load imbalance the plan's LPT assignment leaves (BASELINE.json north_star: "persistent tile scheduler that
 * balances work across SMs regardless of sequence-length skew"; the paper's Fig. 9 / Fig. 10 analogue inside one GPU). */
int arachne_plan_cta_times(const arachne_plan* plan, int kernel, double* start_us, double* end_us, int n, int* n_ctas);

/* Forward.  q, k, v: raw bf16 [N,H,D] (Q, K pre-norm, pre-RoPE).  Writes o (bf16 [N,H,D])
 * and lse (fp32 [H,N]).  workspace: >= arachne_workspace_bytes(plan, 0), 256-byte aligned
 * recommended (16 required); its contents are scratch.  In one-shard plans V is read IN PLACE by the main kernel
 * (tensor-map TMA, encoded per call from the v pointer: v must stay valid and unmodified until the call has run on the
 * stream, like every input), Q and K by the in-call prologue (csrc/prep.cuh). */
int arachne_varlen_attn_fwd(const arachne_plan* plan, const void* q, const void* k, const void* v,
                            const float* gamma_q, const float* gamma_k, void* o, float* lse,
                            void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Forward for call sites that have NO device memory to offer as a workspace and no way of getting any.
 *
 * Who that is.  arachne_varlen_attn_fwd wants a caller-owned workspace, which in practice means somebody called cudaMalloc
 * (or asked a framework allocator that did).  Some users of this library sit where that is not possible: an attention
 * layer plugged into a training process whose caching allocator has already reserved the GPU's memory, so a second,
 * raw cudaMalloc from inside the layer fails or forces the framework to give its cache back; a C host that is handed
 * tensor pointers by its embedder and nothing else — no allocator handle, no permission to create device buffers of its
 * own; and per-layer call sites in a steady-state step loop, where cudaMalloc / cudaFree are banned because they
 * serialise the whole device behind them.  Such a caller still has a plan (built once at set-up by whoever owns the
 * process, where allocation is allowed) and the tensors q, k, v, o, lse.  This call needs nothing more.
 *
 * What it does.  The same two launches as arachne_varlen_attn_fwd (prologue + fwd_kernel, same results), except that the
 * scratch they share — the workspace header and the Q^ / K^ operand images — lives in an array compiled into the library
 * (a file-scope `static __device__` array of ARACHNE_BUILTIN_SCRATCH_BYTES bytes).  Every GPU on which the library's code
 * gets loaded carries those bytes until the process exits, whether or not this call is ever made; that is why the limit
 * is kept small.  The call itself performs no cudaMalloc, cudaFree or any other allocating routine.
 *
 * Limit.  arachne_workspace_bytes(plan, 0) must be <= ARACHNE_BUILTIN_SCRATCH_BYTES (32 MiB: about 65 000 (token, head)
 * rows at head_dim 128, twice that at 64, counting each sequence rounded up to whole 128-token tiles).  Anything larger
 * is refused with ARACHNE_ERR_BUILTIN_SCRATCH before a kernel is launched, and arachne_last_error_message says how many
 * bytes were needed; use arachne_varlen_attn_fwd with a workspace for those.
 *
 * First call on a device.  The device address of the array is looked up (cudaGetSymbolAddress) the first time this
 * function runs on a given device, with that device current, and remembered.  The look-up may make the CUDA runtime load
 * the library's device code, so make one call on each device during set-up, before any stream capture is begun;
 * later calls only read the remembered address.  The plan's device must be the current device (else ARACHNE_ERR_BAD_PARAM).
 *
 * Sharing.  There is ONE array per device, used by every call of this function from every plan and thread in the process.
 * It still holds whatever the previous call left in it; the words that have to start at zero (the workspace header:
 * logit bound, dynamic work counters) are cleared on the stream at the start of every call, everything else is
 * overwritten before it is read.  Two calls whose kernels can overlap on the GPU — different streams, or different host
 * threads — would write over each other's operand images: keep all calls on a device ordered on one stream (or by
 * events).  arachne_varlen_attn_fwd with separate workspaces remains the way to run forwards concurrently.
 *
 * Arguments, layouts, alignment and every other status as arachne_varlen_attn_fwd (one-shard plans only). */
#define ARACHNE_BUILTIN_SCRATCH_BYTES (32u << 20)
int arachne_varlen_attn_fwd_noalloc(const arachne_plan* plan, const void* q, const void* k, const void* v,
                                    const float* gamma_q, const float* gamma_k, void* o, float* lse,
                                    void* cuda_stream);

/* Backward.  Needs the o and lse that fwd produced for the same inputs and plan, and d_o
 * (bf16 [N,H,D]).  Writes dq, dk (gradients w.r.t. the RAW q, k) and dv, all bf16 [N,H,D].
 * With ARACHNE_FLAG_DETERMINISTIC the result is bit-identical from run to run on the same
 * device and plan: the fused kernel's dQ partial tiles are reduced as int32 FIXED POINT (scale = a power of two per
 * (token, head) query row from a rigorous bound on every partial sum of that row, 2 |dO_i| max|V| max|k~|: no overflow in any
 * order), and integer addition is associative, so the order in which the CTAs' reductions reach L2 cannot matter (DESIGN.md
 * §5); everything else has one owner per output tile.  Same speed as the default mode; the quantum is ~2^-13 .. 2^-17 of a
 * typical element of the same row, however large or small that row's dO is (an outlying V row 2^k above typical costs every
 * row of its (sequence, head) group k of those bits).  The bound presumes lse is the forward's own; a dQ row that saw a
 * non-finite or out-of-range partial comes back as NaN (never silently wrapped or zeroed).
 * V and d_o are read in place by tensor-map TMA as in
 * the forward (one-shard plans). */
int arachne_varlen_attn_bwd(const arachne_plan* plan, const void* q, const void* k, const void* v,
                            const float* gamma_q, const float* gamma_k, const void* o,
                            const float* lse, const void* d_o, void* dq, void* dk, void* dv,
                            void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Backward that ALSO returns the gradients of the RMSNorm weights (DESIGN.md reading
 * R22): dgamma_q[d] = sum over all tokens n and heads h of (R^T dq~)[n,h,d] * Q[n,h,d] * r_q[n,h], where
 * dq~ is the gradient w.r.t. the normed + rotated query, R^T the inverse rotation and r = rsqrt(mean(x^2) +
 * eps); likewise dgamma_k.  fp32 [D] DEVICE, fully overwritten; either may be NULL (not computed).  gamma is
 * shared by all heads (R1), so the sum runs over heads too.  With ARACHNE_FLAG_NO_NORM both are zero.  The
 * sum is taken in a fixed order (per-block partials, then block order), so given the same dq~/dk~ it is
 * bit-reproducible.  Enqueues one more (tiny) kernel than arachne_varlen_attn_bwd; everything else is
 * identical, and arachne_workspace_bytes(plan, 1) covers it. */
int arachne_varlen_attn_bwd_dgamma(const arachne_plan* plan, const void* q, const void* k, const void* v,
                                   const float* gamma_q, const float* gamma_k, const void* o,
                                   const float* lse, const void* d_o, void* dq, void* dk, void* dv,
                                   float* dgamma_q, float* dgamma_k,
                                   void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Forward / backward on token-range-sharded tensors (plan from arachne_plan_create_sharded; a plan from
 * arachne_plan_create[_joint] is the 1-shard case and is accepted too).  Every `const void* const* x` is a HOST
 * array of num_shards DEVICE pointers, x[r] = base of shard r ([n_r, total_heads, D] bf16, 16-byte aligned;
 * may be NULL iff shard r is empty).  Same semantics, workspace and stream rules as the plain calls;
 * dgamma_q / dgamma_k may be NULL. */
int arachne_varlen_attn_fwd_sharded(const arachne_plan* plan, const void* const* q, const void* const* k,
                                    const void* const* v, const float* gamma_q, const float* gamma_k,
                                    void* const* o, float* lse, void* workspace, size_t workspace_bytes,
                                    void* cuda_stream);
int arachne_varlen_attn_bwd_sharded(const arachne_plan* plan, const void* const* q, const void* const* k,
                                    const void* const* v, const float* gamma_q, const float* gamma_k,
                                    const void* const* o, const float* lse, const void* const* d_o,
                                    void* const* dq, void* const* dk, void* const* dv,
                                    float* dgamma_q, float* dgamma_k,
                                    void* workspace, size_t workspace_bytes, void* cuda_stream);

/* CONTEXT PARALLELISM ("CP ... partitions the sequence ... K/V ring") without a
 * ring: the packed batch is split by token range into num_shards buffers exactly as for arachne_plan_create_sharded
 * (shard r = [n_r, num_heads, D], ALL heads), and rank `rank` computes, for ALL heads, the attention of ITS query
 * tokens [shard_starts[rank], shard_starts[rank+1]) against all keys of their sequences — K and V rows of the other
 * ranks are read straight from their shards (peer memory; the all-gather of K/V is these loads).
 *   forward : arachne_varlen_attn_fwd_sharded with this plan; only O rows of the rank's own tokens are written (so only
 *             o[rank] is touched) and only those columns of the LOCAL lse [num_heads, N] are defined.
 *   backward: (1) arachne_varlen_attn_bwd_cp_partial on every rank: finishes dQ for the rank's own rows (writes
 *             dq[rank]) and leaves dk~, dV as fp32 PARTIAL sums over the rank's query rows in dk_partial, dv_partial
 *             (fp32 [N, num_heads, D] DEVICE buffers that the other ranks can read; rows of sequences the rank does
 *             not touch are left unwritten);  (2) after a barrier, arachne_cp_reduce on every rank: for the rank's own
 *             key tokens adds the partials of the contributing ranks in RANK ORDER (fixed order; the reduce-scatter
 *             is these peer loads), applies un-RoPE + RMSNorm backward, and writes dk[rank], dv[rank] (bf16) and
 *             dgamma_k (this rank's part; all-reduce it).  dgamma_q comes from step (1) (this rank's part).
 * Sequences may straddle the cuts; rows of a boundary tile that belong to another rank are masked (P = 0), so nothing
 * is counted twice.  With ARACHNE_FLAG_DETERMINISTIC the whole backward is bit-reproducible here too: dQ by the fixed-point
 * reduction, dK / dV because the partials are added in rank order.
 * Workspace for both backward calls: arachne_workspace_bytes(plan, 1).  A rank may own no tokens (empty shard). */
int arachne_plan_create_cp(arachne_plan** out, const arachne_attn_params* params,
                           const int32_t* cu_seqlens_host, const int32_t* grids_host,
                           const int32_t* text_lens_host, int32_t num_shards,
                           const int32_t* shard_starts_host, int32_t rank);
int arachne_varlen_attn_bwd_cp_partial(const arachne_plan* plan, const void* const* q, const void* const* k,
                                       const void* const* v, const float* gamma_q, const float* gamma_k,
                                       const void* const* o, const float* lse, const void* const* d_o,
                                       void* const* dq, float* dk_partial, float* dv_partial, float* dgamma_q,
                                       void* workspace, size_t workspace_bytes, void* cuda_stream);
/* dk_partials / dv_partials: HOST arrays of num_shards DEVICE pointers (rank r's dk_partial / dv_partial). */
int arachne_cp_reduce(const arachne_plan* plan, const float* const* dk_partials, const float* const* dv_partials,
                      const void* const* k, const float* gamma_k, void* const* dk, void* const* dv,
                      float* dgamma_k, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Peer-memory plumbing for the *_sharded / *_cp calls on one node: CUDA IPC.  arachne_ipc_alloc = cudaMalloc on the
 * current device + cudaIpcGetMemHandle (handle_out: 64 bytes, HOST; send it to the other ranks by any means);
 * arachne_ipc_open maps another PROCESS's allocation into this one (the returned device pointer reaches the owner's HBM
 * over NVLink / NVSwitch when the owner is another GPU; the same GPU works too) — not callable on a handle of this
 * process; arachne_ipc_close unmaps, arachne_ipc_free frees an arachne_ipc_alloc allocation (after every peer closed it).
 * Status codes as everywhere (ARACHNE_ERR_CUDA + arachne_last_error_message on a CUDA failure). */
int arachne_ipc_alloc(size_t bytes, void** dev_ptr, void* handle_out);
int arachne_ipc_open(const void* handle, void** dev_ptr);
int arachne_ipc_close(void* dev_ptr);
int arachne_ipc_free(void* dev_ptr);

/* End-to-end convenience calls with HOST tensors (same layouts, all *_host pointers are host
 * memory; pinned for the copies to overlap the kernels, pageable works but serialises): copy in,
 * run, copy the results back, and return after everything has completed.  Device buffers and two
 * private streams are created by the first host call on a plan and kept until arachne_plan_destroy;
 * dO is uploaded while the forward runs and O, LSE are downloaded while the backward runs.  Not
 * re-entrant per plan.  These are the calls bench.py times for its "e2e" figure. */
int arachne_varlen_attn_fwd_host(const arachne_plan* plan, const void* q_host, const void* k_host,
                                 const void* v_host, const float* gamma_q_host,
                                 const float* gamma_k_host, void* o_host, float* lse_host);
int arachne_varlen_attn_fwd_bwd_host(const arachne_plan* plan, const void* q_host,
                                     const void* k_host, const void* v_host,
                                     const float* gamma_q_host, const float* gamma_k_host,
                                     const void* d_o_host, void* o_host, float* lse_host,
                                     void* dq_host, void* dk_host, void* dv_host);

const char* arachne_status_string(int status);
/* Text of the last CUDA error seen by the calling thread ("" if none). */
const char* arachne_last_error_message(void);

#ifdef __cplusplus
}
#endif
#endif /* ARACHNE_ATTN_H_ */
