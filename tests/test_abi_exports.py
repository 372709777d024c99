"""CPU-only: the C-ABI library builds for sm_100a, loads, and exports every symbol that
include/arachne_attn.h declares; argument validation that needs no device is exercised."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    with open(os.path.join(ROOT, "include", "arachne_attn.h")) as f:
        src = f.read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(arachne_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2607_01701_b200 import build

    lib = ctypes.CDLL(build.build())
    names = _declared_symbols()
    assert "arachne_varlen_attn_fwd" in names and "arachne_varlen_attn_bwd" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/arachne_attn.h but not exported"
    from paper_2607_01701_b200 import binding

    assert sorted(binding.EXPORTS) == names
    # ABI version handshake (binding.py refuses a library whose struct layout it does not marshal for)
    with open(os.path.join(ROOT, "include", "arachne_attn.h")) as f:
        declared = int(re.search(r"#define\s+ARACHNE_ABI_VERSION\s+(\d+)", f.read()).group(1))
    lib.arachne_abi_version.restype = ctypes.c_int
    lib.arachne_attn_params_size.restype = ctypes.c_size_t
    assert lib.arachne_abi_version() == declared == binding.ABI_VERSION
    assert lib.arachne_attn_params_size() == ctypes.sizeof(binding.AttnParams) == 72


def test_status_strings_and_validation_without_device():
    from paper_2607_01701_b200 import binding

    lib = binding._lib
    for s in range(0, 16):
        assert lib.arachne_status_string(s).decode() not in ("", "unknown status")
    assert lib.arachne_status_string(99).decode() == "unknown status"
    assert lib.arachne_workspace_bytes(None, 0) == 0
    h = ctypes.c_void_p()
    p = binding.AttnParams()
    assert lib.arachne_plan_create(ctypes.byref(h), None, None, None) == 1            # null pointer
    cu = (ctypes.c_int32 * 2)(0, 64)
    gr = (ctypes.c_int32 * 3)(1, 8, 8)
    p.num_seqs, p.total_tokens, p.num_heads, p.head_dim = 1, 64, 2, 96
    p.rope_dims[:] = [32, 32, 32]
    p.rope_theta, p.rms_eps = 10000.0, 1e-6
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr) == 2     # bad head_dim
    p.head_dim = 64
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr) == 3     # rope dims do not sum to D
    p.rope_dims[:] = [16, 24, 24]
    cu2 = (ctypes.c_int32 * 2)(1, 64)
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu2, gr) == 4    # cu_seqlens[0] != 0
    p.total_tokens = 65
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr) == 6     # total tokens
    p.total_tokens = 64
    gr2 = (ctypes.c_int32 * 3)(1, 8, 9)
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == 5    # grid mismatch
    assert lib.arachne_varlen_attn_fwd(None, None, None, None, None, None, None, None, None, 0, None) == 1
    assert lib.arachne_varlen_attn_fwd_noalloc(None, None, None, None, None, None, None, None, None) == 1
    # 32-bit row indices on the device: tokens x heads must stay below 2^31 (rejected before any CUDA call)
    big = binding.AttnParams()
    big.num_seqs, big.total_tokens, big.num_heads, big.head_dim = 1, 2 ** 27, 16, 64
    big.rope_dims[:] = [16, 24, 24]
    big.rope_theta, big.rms_eps = 10000.0, 1e-6
    cu_big = (ctypes.c_int32 * 2)(0, 2 ** 27)
    gr_big = (ctypes.c_int32 * 3)(2 ** 27, 1, 1)
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(big), cu_big, gr_big) == 11
    # envelope (arachne_attn.h "Verified envelope"): an explicit softmax_scale with scale*sqrt(D) > 1 is refused on the host
    # unless the caller passes ARACHNE_FLAG_WIDE_LOGITS (then validation goes on: here to the grid check)
    p.softmax_scale = 0.2
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == binding.ERR_LOGIT_RANGE
    p.flags = binding.FLAG_WIDE_LOGITS
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == 5
    p.flags = 256                                                                      # unknown flag bit
    assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == 12
    # every flag the header declares is accepted (validation goes on to the grid check) ...
    p.softmax_scale = 0.0
    for f in (binding.FLAG_DETERMINISTIC, binding.FLAG_NO_NORM, binding.FLAG_NO_ROPE, binding.FLAG_WIDE_LOGITS, binding.FLAG_FWD_CTA_PAIRS,
              binding.FLAG_IMAGE_COPIES, binding.FLAG_FWD_MULTICAST, binding.FLAG_FWD_FUSED_Q, 255):
        p.flags = f
        assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == 5, f
    # ... and the token strides of Q / K / V (elements): multiples of 8, >= num_heads * head_dim (no overlapping rows)
    p.flags = 0
    for name in ("q_stride", "k_stride", "v_stride"):
        for bad in (2 * 64 - 8, 2 * 64 + 4, -128):
            setattr(p, name, bad)
            assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == 12, (name, bad)
        setattr(p, name, 3 * 2 * 64)                                                    # a slice of a fused [N, 3, H, D] projection
        assert lib.arachne_plan_create(ctypes.byref(h), ctypes.byref(p), cu, gr2) == 5
        setattr(p, name, 0)


def test_binding_rejects_tensors_the_c_side_cannot_check():
    """dtype, device, contiguity and shape are checked by the marshalling layer (the C ABI sees only pointers)."""
    import pytest
    import torch
    from paper_2607_01701_b200 import binding

    good = torch.zeros(6, 2, 8, dtype=torch.bfloat16)
    binding._want(good, "q", torch.bfloat16, (6, 2, 8), device="cpu")
    binding._want(None, "gamma_q", torch.float32, (8,), device="cpu", optional=True)
    for bad in (good.float(), good[:, :1], good.transpose(0, 1), torch.zeros(6, 2, 4, dtype=torch.bfloat16)):
        with pytest.raises(TypeError):
            binding._want(bad, "q", torch.bfloat16, (6, 2, 8), device="cpu")
    with pytest.raises(TypeError):
        binding._want(good, "q", torch.bfloat16, (6, 2, 8), device="cuda")      # a host tensor where a device one is needed
    with pytest.raises(TypeError):
        binding._want(None, "q", torch.bfloat16, (6, 2, 8))
