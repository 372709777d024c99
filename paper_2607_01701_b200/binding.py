"""Thin ctypes binding over libarachne_attn.so (include/arachne_attn.h) — argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  torch is used for device
memory and streams.  There is NO fallback: importing this module raises if the library has not
been built (python -m paper_2607_01701_b200.build), and every call raises on a non-zero status.
"""
from __future__ import annotations

import ctypes
import os

import torch

_LIB_PATH = os.environ.get("ARACHNE_ATTN_LIB") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "libarachne_attn.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(
        f"{_LIB_PATH} is missing: build it with `python -m paper_2607_01701_b200.build` "
        "(nvcc, sm_100a). There is no CPU fallback.")
_lib = ctypes.CDLL(_LIB_PATH)

FLAG_DETERMINISTIC, FLAG_NO_NORM, FLAG_NO_ROPE, FLAG_WIDE_LOGITS, FLAG_FWD_CTA_PAIRS, FLAG_IMAGE_COPIES, FLAG_FWD_MULTICAST, FLAG_FWD_FUSED_Q = 1, 2, 4, 8, 16, 32, 64, 128
ERR_LOGIT_RANGE = 14
ERR_BUILTIN_SCRATCH = 15
BUILTIN_SCRATCH_BYTES = 32 << 20      # ARACHNE_BUILTIN_SCRATCH_BYTES (include/arachne_attn.h)

EXPORTS = [
    "arachne_plan_create", "arachne_plan_destroy", "arachne_workspace_bytes", "arachne_num_launches",
    "arachne_varlen_attn_fwd", "arachne_varlen_attn_bwd", "arachne_varlen_attn_fwd_host",
    "arachne_varlen_attn_fwd_bwd_host", "arachne_status_string", "arachne_last_error_message",
    "arachne_kernel_name", "arachne_plan_enable_profiling", "arachne_plan_kernel_times",
    "arachne_plan_create_joint", "arachne_varlen_attn_bwd_dgamma",
    "arachne_plan_create_sharded", "arachne_varlen_attn_fwd_sharded", "arachne_varlen_attn_bwd_sharded",
    "arachne_plan_create_cp", "arachne_varlen_attn_bwd_cp_partial", "arachne_cp_reduce",
    "arachne_ipc_alloc", "arachne_ipc_open", "arachne_ipc_close", "arachne_ipc_free", "arachne_plan_cta_times",
    "arachne_plan_logit_status", "arachne_varlen_attn_fwd_noalloc", "arachne_abi_version", "arachne_attn_params_size",
]


class AttnParams(ctypes.Structure):
    _fields_ = [
        ("num_seqs", ctypes.c_int32), ("total_tokens", ctypes.c_int32), ("num_heads", ctypes.c_int32),
        ("head_dim", ctypes.c_int32), ("rope_dims", ctypes.c_int32 * 3), ("rope_theta", ctypes.c_float),
        ("rms_eps", ctypes.c_float), ("softmax_scale", ctypes.c_float), ("flags", ctypes.c_int32),
        ("q_stride", ctypes.c_int64), ("k_stride", ctypes.c_int64), ("v_stride", ctypes.c_int64),
    ]


ABI_VERSION = 3      # ARACHNE_ABI_VERSION of the header this file marshals for (include/arachne_attn.h)
if not hasattr(_lib, "arachne_abi_version"):
    raise ImportError(f"{_LIB_PATH} predates arachne_abi_version(): rebuild it (python -m paper_2607_01701_b200.build)")
_lib.arachne_abi_version.restype = ctypes.c_int
_lib.arachne_attn_params_size.restype = ctypes.c_size_t
if _lib.arachne_abi_version() != ABI_VERSION or _lib.arachne_attn_params_size() != ctypes.sizeof(AttnParams):
    # a stale .so would read q_stride / k_stride / v_stride (or whatever came later) past the end of the struct we pass
    raise ImportError(f"{_LIB_PATH}: ABI version {_lib.arachne_abi_version()} / params size {_lib.arachne_attn_params_size()}, "
                      f"binding.py expects {ABI_VERSION} / {ctypes.sizeof(AttnParams)}: rebuild the library")

_vp, _i32p, _fp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int32), ctypes.c_void_p
_lib.arachne_plan_create.restype = ctypes.c_int
_lib.arachne_plan_create.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(AttnParams), _i32p, _i32p]
_lib.arachne_plan_create_joint.restype = ctypes.c_int
_lib.arachne_plan_create_joint.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(AttnParams), _i32p, _i32p, _i32p]
_lib.arachne_plan_create_sharded.restype = ctypes.c_int
_lib.arachne_plan_create_sharded.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(AttnParams), _i32p, _i32p, _i32p,
                                             ctypes.c_int32, _i32p, ctypes.c_int32, ctypes.c_int32]
_lib.arachne_plan_destroy.restype = None
_lib.arachne_plan_destroy.argtypes = [_vp]
_lib.arachne_workspace_bytes.restype = ctypes.c_size_t
_lib.arachne_workspace_bytes.argtypes = [_vp, ctypes.c_int]
_lib.arachne_num_launches.restype = ctypes.c_int
_lib.arachne_num_launches.argtypes = [_vp, ctypes.c_int]
_lib.arachne_varlen_attn_fwd.restype = ctypes.c_int
_lib.arachne_varlen_attn_fwd.argtypes = [_vp] * 8 + [_vp, ctypes.c_size_t, _vp]
_lib.arachne_varlen_attn_fwd_noalloc.restype = ctypes.c_int
_lib.arachne_varlen_attn_fwd_noalloc.argtypes = [_vp] * 8 + [_vp]
_lib.arachne_varlen_attn_bwd.restype = ctypes.c_int
_lib.arachne_varlen_attn_bwd.argtypes = [_vp] * 12 + [_vp, ctypes.c_size_t, _vp]
_lib.arachne_varlen_attn_bwd_dgamma.restype = ctypes.c_int
_lib.arachne_varlen_attn_bwd_dgamma.argtypes = [_vp] * 14 + [_vp, ctypes.c_size_t, _vp]
_vpp = ctypes.POINTER(ctypes.c_void_p)
_lib.arachne_varlen_attn_fwd_sharded.restype = ctypes.c_int
_lib.arachne_varlen_attn_fwd_sharded.argtypes = [_vp, _vpp, _vpp, _vpp, _vp, _vp, _vpp, _vp, _vp, ctypes.c_size_t, _vp]
_lib.arachne_varlen_attn_bwd_sharded.restype = ctypes.c_int
_lib.arachne_varlen_attn_bwd_sharded.argtypes = [_vp, _vpp, _vpp, _vpp, _vp, _vp, _vpp, _vp, _vpp, _vpp, _vpp, _vpp,
                                                 _vp, _vp, _vp, ctypes.c_size_t, _vp]
_lib.arachne_plan_create_cp.restype = ctypes.c_int
_lib.arachne_plan_create_cp.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(AttnParams), _i32p, _i32p, _i32p,
                                        ctypes.c_int32, _i32p, ctypes.c_int32]
_lib.arachne_varlen_attn_bwd_cp_partial.restype = ctypes.c_int
_lib.arachne_varlen_attn_bwd_cp_partial.argtypes = [_vp, _vpp, _vpp, _vpp, _vp, _vp, _vpp, _vp, _vpp, _vpp, _vp, _vp, _vp,
                                                    _vp, ctypes.c_size_t, _vp]
_lib.arachne_cp_reduce.restype = ctypes.c_int
_lib.arachne_cp_reduce.argtypes = [_vp, _vpp, _vpp, _vpp, _vp, _vpp, _vpp, _vp, _vp, ctypes.c_size_t, _vp]
_lib.arachne_varlen_attn_fwd_host.restype = ctypes.c_int
_lib.arachne_varlen_attn_fwd_host.argtypes = [_vp] * 8
_lib.arachne_varlen_attn_fwd_bwd_host.restype = ctypes.c_int
_lib.arachne_varlen_attn_fwd_bwd_host.argtypes = [_vp] * 12
_lib.arachne_status_string.restype = ctypes.c_char_p
_lib.arachne_status_string.argtypes = [ctypes.c_int]
_lib.arachne_last_error_message.restype = ctypes.c_char_p
_lib.arachne_kernel_name.restype = ctypes.c_char_p
_lib.arachne_kernel_name.argtypes = [ctypes.c_int, ctypes.c_int]
_lib.arachne_plan_enable_profiling.restype = ctypes.c_int
_lib.arachne_plan_enable_profiling.argtypes = [_vp, ctypes.c_int]
_lib.arachne_plan_kernel_times.restype = ctypes.c_int
_lib.arachne_plan_kernel_times.argtypes = [_vp, ctypes.c_int, ctypes.POINTER(ctypes.c_float), ctypes.c_int,
                                           ctypes.POINTER(ctypes.c_int)]


_lib.arachne_ipc_alloc.restype = ctypes.c_int
_lib.arachne_ipc_alloc.argtypes = [ctypes.c_size_t, ctypes.POINTER(_vp), ctypes.c_char_p]
_lib.arachne_ipc_open.restype = ctypes.c_int
_lib.arachne_ipc_open.argtypes = [ctypes.c_char_p, ctypes.POINTER(_vp)]
_lib.arachne_ipc_close.restype = ctypes.c_int
_lib.arachne_ipc_close.argtypes = [_vp]
_lib.arachne_ipc_free.restype = ctypes.c_int
_lib.arachne_ipc_free.argtypes = [_vp]


_lib.arachne_plan_cta_times.restype = ctypes.c_int
_lib.arachne_plan_cta_times.argtypes = [_vp, ctypes.c_int, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                        ctypes.c_int, ctypes.POINTER(ctypes.c_int)]


_lib.arachne_plan_logit_status.restype = ctypes.c_int
_lib.arachne_plan_logit_status.argtypes = [_vp, ctypes.POINTER(ctypes.c_float)]


class ArachneError(RuntimeError):
    def __init__(self, status: int):
        self.status = status
        msg = _lib.arachne_status_string(status).decode()
        detail = _lib.arachne_last_error_message().decode()
        super().__init__(f"arachne status {status}: {msg}" + (f" ({detail})" if status in (10, ERR_BUILTIN_SCRATCH) and detail else ""))


def _check(status: int):
    if status != 0:
        raise ArachneError(status)


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _want(t, name, dtype, shape=None, device="cuda", optional=False, tok_stride=0):
    """The C side can only check alignment: a non-contiguous view (a slice of a fused QKV projection), a wrong dtype or a
    CPU tensor would silently give wrong results or fault, so the marshalling layer refuses them here."""
    if t is None:
        if optional:
            return
        raise TypeError(f"{name}: tensor required")
    if t.device.type != device:
        raise TypeError(f"{name}: expected a {device} tensor, got {t.device}")
    if t.dtype != dtype:
        raise TypeError(f"{name}: expected {dtype}, got {t.dtype}")
    if tok_stride:
        # a token-strided view declared at plan creation (q_stride / k_stride / v_stride): heads and head_dim stay dense
        if shape is None or len(shape) != 3 or tuple(t.stride()) != (tok_stride, shape[2], 1):
            raise TypeError(f"{name}: expected strides ({tok_stride}, D, 1) as declared to the plan, got {tuple(t.stride())}")
    elif not t.is_contiguous():
        raise TypeError(f"{name}: must be contiguous (or declare its token stride to the plan: q_stride / k_stride / v_stride)")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise TypeError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")


def _want_call(plan, bf16, lse=None, gammas=(), workspace=None, device="cuda"):
    nhd = (plan.N, plan.total_heads, plan.D)
    for name, t in bf16.items():
        _want(t, name, torch.bfloat16, nhd, device, tok_stride=getattr(plan, "in_strides", {}).get(name, 0))
    if lse is not None:
        _want(lse, "lse", torch.float32, (plan.H, plan.N), device)
    for name, t in gammas:
        _want(t, name, torch.float32, (plan.D,), device, optional=True)
    if workspace is not None:
        _want(workspace, "workspace", torch.uint8, None, device)


class Plan:
    """arachne_plan_create[_joint] / arachne_plan_destroy.  text_lens [B] (optional): trailing text tokens of
    each sequence (arachne_plan_create_joint).  shard_starts [k+1] (+ total_heads, head_offset): token-range
    sharding of the raw tensors for the fused-All-to-All Ulysses calls (arachne_plan_create_sharded); num_heads
    is then the LOCAL head count."""

    def __init__(self, cu_seqlens, grids, num_heads, head_dim, rope_dims, rope_theta=10000.0, rms_eps=1e-6,
                 softmax_scale=0.0, flags=0, text_lens=None, shard_starts=None, total_heads=None, head_offset=0, cp_rank=None,
                 q_stride=0, k_stride=0, v_stride=0):
        cu = [int(x) for x in cu_seqlens]
        gr = [int(x) for g in grids for x in g]
        self.params = AttnParams()
        self.params.num_seqs = len(cu) - 1
        self.params.total_tokens = cu[-1] if cu else 0
        self.params.num_heads = num_heads
        self.params.head_dim = head_dim
        self.params.rope_dims[:] = [int(x) for x in rope_dims]
        self.params.rope_theta = rope_theta
        self.params.rms_eps = rms_eps
        self.params.softmax_scale = softmax_scale
        self.params.flags = flags
        # token strides (elements) of strided Q / K / V views, e.g. slices of a fused [N, 3, H, D] projection; 0 = contiguous
        self.params.q_stride, self.params.k_stride, self.params.v_stride = int(q_stride), int(k_stride), int(v_stride)
        self.in_strides = {"q": int(q_stride), "k": int(k_stride), "v": int(v_stride)}
        self._h = _vp()
        cu_arr = (ctypes.c_int32 * len(cu))(*cu)
        gr_arr = (ctypes.c_int32 * max(len(gr), 1))(*gr)
        self.num_shards = 1
        if shard_starts is not None:
            ss = [int(x) for x in shard_starts]
            self.num_shards = len(ss) - 1
            ss_arr = (ctypes.c_int32 * len(ss))(*ss)
            tl_arr = None
            if text_lens is not None:
                tl = [int(x) for x in text_lens]
                tl_arr = (ctypes.c_int32 * max(len(tl), 1))(*tl)
            if cp_rank is not None:      # context parallelism: arachne_plan_create_cp
                _check(_lib.arachne_plan_create_cp(ctypes.byref(self._h), ctypes.byref(self.params), cu_arr, gr_arr, tl_arr,
                                                   self.num_shards, ss_arr, int(cp_rank)))
            else:
                _check(_lib.arachne_plan_create_sharded(ctypes.byref(self._h), ctypes.byref(self.params), cu_arr, gr_arr, tl_arr,
                                                        self.num_shards, ss_arr, int(total_heads or num_heads), int(head_offset)))
        elif text_lens is None:
            _check(_lib.arachne_plan_create(ctypes.byref(self._h), ctypes.byref(self.params), cu_arr, gr_arr))
        else:
            tl = [int(x) for x in text_lens]
            tl_arr = (ctypes.c_int32 * max(len(tl), 1))(*tl)
            _check(_lib.arachne_plan_create_joint(ctypes.byref(self._h), ctypes.byref(self.params), cu_arr, gr_arr, tl_arr))
        self.N, self.H, self.D = self.params.total_tokens, num_heads, head_dim
        self.total_heads = int(total_heads or num_heads)      # heads in the raw tensors (> H for an Ulysses rank's plan)

    def workspace_bytes(self, bwd: bool) -> int:
        return int(_lib.arachne_workspace_bytes(self._h, 1 if bwd else 0))

    def num_launches(self, bwd: bool) -> int:
        return int(_lib.arachne_num_launches(self._h, 1 if bwd else 0))

    def enable_profiling(self, enable=True):
        _check(_lib.arachne_plan_enable_profiling(self._h, 1 if enable else 0))

    def logit_status(self):
        """(status, tau): arachne_plan_logit_status — ERR_LOGIT_RANGE once a forward without FLAG_WIDE_LOGITS saw tau > 1."""
        tau = ctypes.c_float(0.0)
        return int(_lib.arachne_plan_logit_status(self._h, ctypes.byref(tau))), float(tau.value)

    def kernel_times(self, bwd: bool):
        """[(timed interval name, mean ms per call)] over the calls recorded since enable_profiling()."""
        n = 3 if bwd else 2
        ms = (ctypes.c_float * n)()
        calls = ctypes.c_int(0)
        _check(_lib.arachne_plan_kernel_times(self._h, 1 if bwd else 0, ms, n, ctypes.byref(calls)))
        c = max(calls.value, 1)
        return [(_lib.arachne_kernel_name(1 if bwd else 0, i).decode(), ms[i] / c) for i in range(n)], calls.value

    def cta_times(self, bwd: bool):
        """(start_us[], end_us[]) of every CTA of the last fwd_kernel / bwd_fused_kernel launch (arachne_plan_cta_times)."""
        cap = 256
        s, e, n = (ctypes.c_double * cap)(), (ctypes.c_double * cap)(), ctypes.c_int(0)
        _check(_lib.arachne_plan_cta_times(self._h, 1 if bwd else 0, s, e, cap, ctypes.byref(n)))
        return list(s[:n.value]), list(e[:n.value])

    def close(self):
        if self._h:
            _lib.arachne_plan_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _stream_ptr(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def arachne_varlen_attn_fwd(plan: Plan, q, k, v, o, lse, workspace, gamma_q=None, gamma_k=None, stream=None):
    """q,k,v,o: bf16 CUDA [N,H,D]; lse: fp32 CUDA [H,N]; workspace: uint8 CUDA >= plan.workspace_bytes(False)."""
    _want_call(plan, dict(q=q, k=k, v=v, o=o), lse, (("gamma_q", gamma_q), ("gamma_k", gamma_k)), workspace)
    _check(_lib.arachne_varlen_attn_fwd(plan._h, _ptr(q), _ptr(k), _ptr(v), _ptr(gamma_q), _ptr(gamma_k), _ptr(o),
                                        _ptr(lse), _ptr(workspace), workspace.numel() * workspace.element_size(),
                                        _stream_ptr(stream)))


def arachne_varlen_attn_fwd_noalloc(plan: Plan, q, k, v, o, lse, gamma_q=None, gamma_k=None, stream=None):
    """The forward for callers with no workspace to give: same tensors as arachne_varlen_attn_fwd, no workspace argument.

    Meant for code that cannot obtain device memory where it runs — a layer inside a process whose framework allocator
    already owns the GPU, an embedded C host that is only handed tensor pointers, a step loop where cudaMalloc / cudaFree
    are off limits because they stall the device.  The scratch is a 32 MiB array built into the library
    (BUILTIN_SCRATCH_BYTES), one per GPU, shared by every call: plans whose plan.workspace_bytes(False) exceeds it raise
    ArachneError(ERR_BUILTIN_SCRATCH); calls that could overlap on the GPU (two streams) corrupt each other, so keep them
    on one stream.  Make the first call on each device during set-up (it looks the array's address up).  Nothing is
    allocated here either: o and lse come from the caller."""
    _want_call(plan, dict(q=q, k=k, v=v, o=o), lse, (("gamma_q", gamma_q), ("gamma_k", gamma_k)))
    _check(_lib.arachne_varlen_attn_fwd_noalloc(plan._h, _ptr(q), _ptr(k), _ptr(v), _ptr(gamma_q), _ptr(gamma_k), _ptr(o),
                                                _ptr(lse), _stream_ptr(stream)))


def arachne_varlen_attn_bwd(plan: Plan, q, k, v, o, lse, d_o, dq, dk, dv, workspace, gamma_q=None, gamma_k=None,
                            stream=None):
    _want_call(plan, dict(q=q, k=k, v=v, o=o, d_o=d_o, dq=dq, dk=dk, dv=dv), lse, (("gamma_q", gamma_q), ("gamma_k", gamma_k)), workspace)
    _check(_lib.arachne_varlen_attn_bwd(plan._h, _ptr(q), _ptr(k), _ptr(v), _ptr(gamma_q), _ptr(gamma_k), _ptr(o),
                                        _ptr(lse), _ptr(d_o), _ptr(dq), _ptr(dk), _ptr(dv), _ptr(workspace),
                                        workspace.numel() * workspace.element_size(), _stream_ptr(stream)))


def arachne_varlen_attn_bwd_dgamma(plan: Plan, q, k, v, o, lse, d_o, dq, dk, dv, dgamma_q, dgamma_k, workspace,
                                   gamma_q=None, gamma_k=None, stream=None):
    """As arachne_varlen_attn_bwd, plus dgamma_q, dgamma_k: fp32 CUDA [D] (either may be None)."""
    _want_call(plan, dict(q=q, k=k, v=v, o=o, d_o=d_o, dq=dq, dk=dk, dv=dv), lse,
               (("gamma_q", gamma_q), ("gamma_k", gamma_k), ("dgamma_q", dgamma_q), ("dgamma_k", dgamma_k)), workspace)
    _check(_lib.arachne_varlen_attn_bwd_dgamma(plan._h, _ptr(q), _ptr(k), _ptr(v), _ptr(gamma_q), _ptr(gamma_k), _ptr(o),
                                               _ptr(lse), _ptr(d_o), _ptr(dq), _ptr(dk), _ptr(dv), _ptr(dgamma_q),
                                               _ptr(dgamma_k), _ptr(workspace),
                                               workspace.numel() * workspace.element_size(), _stream_ptr(stream)))


def _ptr_array(shards, n):
    """HOST array of n device pointers from a list of CUDA tensors / integer addresses / None (empty shard)."""
    assert len(shards) == n, f"expected {n} shards, got {len(shards)}"
    vals = [None if s is None else (int(s) if isinstance(s, int) else s.data_ptr()) for s in shards]
    return (ctypes.c_void_p * n)(*vals)


def arachne_varlen_attn_fwd_sharded(plan: Plan, q, k, v, o, lse, workspace, gamma_q=None, gamma_k=None, stream=None):
    """q, k, v, o: lists of plan.num_shards bf16 CUDA tensors [n_r, total_heads, D] (or raw device addresses of peer
    memory); lse: LOCAL fp32 [num_heads, N]."""
    n = plan.num_shards
    _check(_lib.arachne_varlen_attn_fwd_sharded(plan._h, _ptr_array(q, n), _ptr_array(k, n), _ptr_array(v, n),
                                                _ptr(gamma_q), _ptr(gamma_k), _ptr_array(o, n), _ptr(lse), _ptr(workspace),
                                                workspace.numel() * workspace.element_size(), _stream_ptr(stream)))


def arachne_varlen_attn_bwd_sharded(plan: Plan, q, k, v, o, lse, d_o, dq, dk, dv, workspace, dgamma_q=None, dgamma_k=None,
                                    gamma_q=None, gamma_k=None, stream=None):
    n = plan.num_shards
    _check(_lib.arachne_varlen_attn_bwd_sharded(plan._h, _ptr_array(q, n), _ptr_array(k, n), _ptr_array(v, n),
                                                _ptr(gamma_q), _ptr(gamma_k), _ptr_array(o, n), _ptr(lse),
                                                _ptr_array(d_o, n), _ptr_array(dq, n), _ptr_array(dk, n), _ptr_array(dv, n),
                                                _ptr(dgamma_q), _ptr(dgamma_k), _ptr(workspace),
                                                workspace.numel() * workspace.element_size(), _stream_ptr(stream)))


def arachne_varlen_attn_bwd_cp_partial(plan: Plan, q, k, v, o, lse, d_o, dq, dk_partial, dv_partial, workspace, dgamma_q=None,
                                       gamma_q=None, gamma_k=None, stream=None):
    """Context parallelism, step 1: dq[rank] finished; dk_partial, dv_partial: fp32 CUDA [N,H,D] (this rank's partials)."""
    n = plan.num_shards
    _check(_lib.arachne_varlen_attn_bwd_cp_partial(plan._h, _ptr_array(q, n), _ptr_array(k, n), _ptr_array(v, n),
                                                   _ptr(gamma_q), _ptr(gamma_k), _ptr_array(o, n), _ptr(lse),
                                                   _ptr_array(d_o, n), _ptr_array(dq, n), _ptr(dk_partial), _ptr(dv_partial),
                                                   _ptr(dgamma_q), _ptr(workspace),
                                                   workspace.numel() * workspace.element_size(), _stream_ptr(stream)))


def arachne_cp_reduce(plan: Plan, dk_partials, dv_partials, k, dk, dv, workspace, dgamma_k=None, gamma_k=None, stream=None):
    """Context parallelism, step 2: dk_partials / dv_partials are lists of every rank's partial buffers."""
    n = plan.num_shards
    _check(_lib.arachne_cp_reduce(plan._h, _ptr_array(dk_partials, n), _ptr_array(dv_partials, n), _ptr_array(k, n),
                                  _ptr(gamma_k), _ptr_array(dk, n), _ptr_array(dv, n), _ptr(dgamma_k), _ptr(workspace),
                                  workspace.numel() * workspace.element_size(), _stream_ptr(stream)))


def arachne_varlen_attn_fwd_host(plan: Plan, q, k, v, o, lse, gamma_q=None, gamma_k=None):
    """Same as fwd but every tensor is a HOST (CPU, preferably pinned) tensor; copies are inside the call."""
    _want_call(plan, dict(q=q, k=k, v=v, o=o), lse, (("gamma_q", gamma_q), ("gamma_k", gamma_k)), device="cpu")
    _check(_lib.arachne_varlen_attn_fwd_host(plan._h, _ptr(q), _ptr(k), _ptr(v), _ptr(gamma_q), _ptr(gamma_k),
                                             _ptr(o), _ptr(lse)))


def arachne_varlen_attn_fwd_bwd_host(plan: Plan, q, k, v, d_o, o, lse, dq, dk, dv, gamma_q=None, gamma_k=None):
    _want_call(plan, dict(q=q, k=k, v=v, o=o, d_o=d_o, dq=dq, dk=dk, dv=dv), lse, (("gamma_q", gamma_q), ("gamma_k", gamma_k)),
               device="cpu")
    _check(_lib.arachne_varlen_attn_fwd_bwd_host(plan._h, _ptr(q), _ptr(k), _ptr(v), _ptr(gamma_q), _ptr(gamma_k),
                                                 _ptr(d_o), _ptr(o), _ptr(lse), _ptr(dq), _ptr(dk), _ptr(dv)))


# ---- convenience wrappers that allocate outputs / workspace with torch (plumbing only)
def plan_for(st, flags=0, **kw) -> Plan:
    return Plan(st["cu_seqlens"], st["grids"], st["H"], st["D"], st["rope_dims"], flags=flags,
                text_lens=st.get("text_lens"), **kw)


def forward(plan: Plan, q, k, v, gamma_q=None, gamma_k=None, workspace=None):
    o = torch.empty_like(q)
    lse = torch.empty((plan.H, plan.N), dtype=torch.float32, device=q.device)
    ws = workspace if workspace is not None else torch.empty(plan.workspace_bytes(False), dtype=torch.uint8, device=q.device)
    arachne_varlen_attn_fwd(plan, q, k, v, o, lse, ws, gamma_q, gamma_k)
    return o, lse


def backward(plan: Plan, q, k, v, o, lse, d_o, gamma_q=None, gamma_k=None, workspace=None, with_dgamma=False):
    """Returns (dq, dk, dv) or, with_dgamma, (dq, dk, dv, dgamma_q, dgamma_k)."""
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(v)
    ws = workspace if workspace is not None else torch.empty(plan.workspace_bytes(True), dtype=torch.uint8, device=q.device)
    if not with_dgamma:
        arachne_varlen_attn_bwd(plan, q, k, v, o, lse, d_o, dq, dk, dv, ws, gamma_q, gamma_k)
        return dq, dk, dv
    dgq = torch.empty(plan.D, dtype=torch.float32, device=q.device)
    dgk = torch.empty(plan.D, dtype=torch.float32, device=q.device)
    arachne_varlen_attn_bwd_dgamma(plan, q, k, v, o, lse, d_o, dq, dk, dv, dgq, dgk, ws, gamma_q, gamma_k)
    return dq, dk, dv, dgq, dgk


# ---- CUDA IPC plumbing (peer shards on one node)
def ipc_alloc(nbytes: int):
    """-> (device address, 64-byte handle).  cudaMalloc on the current device; free with ipc_free."""
    ptr, handle = _vp(), ctypes.create_string_buffer(64)
    _check(_lib.arachne_ipc_alloc(nbytes, ctypes.byref(ptr), handle))
    return int(ptr.value), handle.raw


def ipc_open(handle: bytes) -> int:
    ptr = _vp()
    _check(_lib.arachne_ipc_open(handle, ctypes.byref(ptr)))
    return int(ptr.value)


def ipc_close(addr: int):
    _check(_lib.arachne_ipc_close(_vp(addr)))


def ipc_free(addr: int):
    _check(_lib.arachne_ipc_free(_vp(addr)))


class _RawCuda:
    """__cuda_array_interface__ view of raw device memory, so that torch can wrap it without a copy."""

    def __init__(self, addr, shape, typestr):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (addr, False), "version": 3}


def tensor_from_address(addr: int, shape, dtype):
    """torch tensor over raw device memory (bf16 goes through an int16 view: the array interface has no bf16)."""
    if dtype == torch.bfloat16:
        return torch.as_tensor(_RawCuda(addr, shape, "<i2"), device="cuda").view(torch.bfloat16)
    typestr = {torch.float32: "<f4", torch.uint8: "|u1"}[dtype]
    return torch.as_tensor(_RawCuda(addr, shape, typestr), device="cuda")
