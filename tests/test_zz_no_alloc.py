"""arachne_varlen_attn_fwd_noalloc against the ordinary forward (GPU).

The entry point under test exists for users who cannot get hold of device memory where their code runs: an attention
layer embedded in a training process whose framework allocator has already taken the GPU's memory (a raw cudaMalloc
there fails, or evicts the framework's cache), a C host that is only ever handed tensor pointers by its embedder, and
step loops in which cudaMalloc / cudaFree are forbidden because they hold up the whole device.  Instead of a workspace
argument it uses a 32 MiB array compiled into the library, one per GPU, shared by all calls (include/arachne_attn.h).

What is checked: its O and LSE equal the ordinary forward's (same plan, same inputs, workspace from torch) within the
tolerances every parity test here uses (parity_util.TOL), on two calls IN A ROW with different packings and head_dim —
the second call finds the first one's leftovers in the shared array and must not be disturbed by them — then the first
packing once more; and that a packing beyond the limit is refused with ARACHNE_ERR_BUILTIN_SCRATCH before anything runs.

This file is named so that pytest collects it last: under `pytest -x` a failure here cannot hide the other tests.  It
does not depend on them either (nor on a fresh process): whatever earlier calls left in the array is exactly the
situation the entry point is specified for.
"""
import numpy as np
import pytest
import torch

from paper_2607_01701_b200 import inputs

import parity_util as pu

pytestmark = pytest.mark.gpu


def _compare(st, seed_index):
    """One no-alloc forward vs one ordinary forward on the same plan and bytes; returns the worst differences."""
    from paper_2607_01701_b200 import binding

    t = inputs.make_inputs(st, device="cuda")
    plan = binding.plan_for(st)
    assert plan.workspace_bytes(False) <= binding.BUILTIN_SCRATCH_BYTES
    # the caller brings inputs and outputs, nothing else; poison the outputs so that an unwritten row shows
    o = torch.full_like(t["q"], float("nan"))
    lse = torch.full((plan.H, plan.N), float("nan"), dtype=torch.float32, device="cuda")
    binding.arachne_varlen_attn_fwd_noalloc(plan, t["q"], t["k"], t["v"], o, lse)
    o_ref, lse_ref = binding.forward(plan, t["q"], t["k"], t["v"])          # existing path: torch-allocated workspace
    torch.cuda.synchronize()
    got = {"O": pu.to_np(o), "LSE": pu.to_np(lse)}
    ref = {"O": pu.to_np(o_ref), "LSE": pu.to_np(lse_ref)}
    assert np.isfinite(got["O"]).all() and np.isfinite(got["LSE"]).all(), "an output row was left unwritten"
    cu = st["cu_seqlens"]
    worst = dict(O_rel=0.0, O_abs=0.0, LSE_abs=0.0)
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        worst["O_rel"] = max(worst["O_rel"], pu.rel_l2(got["O"][s:e], ref["O"][s:e]))
        worst["O_abs"] = max(worst["O_abs"], float(np.max(np.abs(got["O"][s:e] - ref["O"][s:e]))))
        worst["LSE_abs"] = max(worst["LSE_abs"], float(np.max(np.abs(got["LSE"][:, s:e] - ref["LSE"][:, s:e]))))
    assert worst["O_rel"] <= pu.TOL["O_rel"] and worst["O_abs"] <= pu.TOL["O_abs"], (seed_index, worst)
    assert worst["LSE_abs"] <= pu.TOL["LSE_abs"], (seed_index, worst)
    plan.close()
    return worst


def test_noalloc_forward_matches_the_ordinary_forward_on_consecutive_calls():
    first = inputs.pack([(1, 16, 16), (3, 10, 13)], 3, 128, index=1)          # 256 + 390 tokens (ragged tail), D = 128
    second = inputs.structure("tiny")                                          # BASELINE.json configs[0]: 64 + 200 tokens, D = 64
    third = inputs.pack([(2, 16, 20), (1, 5, 7), (5, 9, 11)], 4, 128, index=5)  # several tiles, a sequence below one tile
    w1 = _compare(first, 1)
    w2 = _compare(second, 2)          # runs on the array as call 1 left it
    w3 = _compare(third, 3)
    w4 = _compare(first, 4)           # and the first packing again, over the leftovers of a different layout
    print("noalloc vs workspace forward:", w1, w2, w3, w4)


def test_noalloc_forward_refuses_packings_beyond_the_builtin_scratch():
    from paper_2607_01701_b200 import binding

    st = inputs.structure("bucket256")          # 15 104 tokens x 24 heads x 128: ~186 MB of operand images, limit is 32 MiB
    plan = binding.plan_for(st)
    assert plan.workspace_bytes(False) > binding.BUILTIN_SCRATCH_BYTES
    q = torch.zeros((plan.N, plan.H, plan.D), dtype=torch.bfloat16, device="cuda")
    o = torch.full_like(q, 7.0)
    lse = torch.full((plan.H, plan.N), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(binding.ArachneError) as ei:
        binding.arachne_varlen_attn_fwd_noalloc(plan, q, q, q, o, lse)
    assert ei.value.status == binding.ERR_BUILTIN_SCRATCH
    assert str(plan.workspace_bytes(False)) in str(ei.value) and str(binding.BUILTIN_SCRATCH_BYTES) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((o == 7.0).all()) and bool((lse == 7.0).all()), "a refused call must not touch the outputs"
    plan.close()
