"""GPU parity tests: the CUDA path (through the C ABI binding) against the fp64 oracle on the same
seeded bytes.  Tolerances are BASELINE.json north_star's: O rel-L2 <= 1e-2 and max-abs <= 2e-2,
LSE max-abs <= 1e-3, dQ/dK/dV rel-L2 <= 2e-2 — checked per tensor AND per sequence (reading R17).
Small cases are compared element by element; the BASELINE.json configs 1-4 on sampled query rows
(exact per row) + the masked-dO backward (exact dK/dV for all key rows) + full-size invariants.
"""
import numpy as np
import pytest
import torch

from paper_2607_01701_b200 import inputs

import parity_util as pu

pytestmark = pytest.mark.gpu


def _np(t):
    return {k: v.float().cpu().numpy().astype(np.float64) for k, v in t.items()}


def _full_case(orc, st, gamma=False, flags=0, oracle_kw=None, plan_kw=None, with_bwd=True):
    t = inputs.make_inputs(st, device="cuda")
    gq = gk = None
    if gamma:
        from paper_2607_01701_b200 import binding
        rng = np.random.default_rng(3)
        gq, gk = (0.5 + rng.random(st["D"])).astype(np.float32), (0.5 + rng.random(st["D"])).astype(np.float32)
        flags |= binding.FLAG_WIDE_LOGITS        # |gamma|inf up to 1.5 each: tau up to 2.25 (arachne_attn.h, "Verified envelope")
    got = pu.run_gpu(st, t, flags=flags, gamma_q=gq, gamma_k=gk, plan_kw=plan_kw, with_bwd=with_bwd)
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"] if with_bwd else None,
                        gamma_q=gq, gamma_k=gk, rope_dims=st["rope_dims"], **(oracle_kw or {}))
    return pu.check_full(st, got, ref, with_bwd=with_bwd), got, t


# ------------------------------------------------------------------ BASELINE.json configs[0]
def test_tiny_config_full(orc):
    w, _, _ = _full_case(orc, inputs.structure("tiny"))
    print("tiny:", w)


# ------------------------------------------------------------------ several tiles + ragged tails, element by element
@pytest.mark.parametrize("grids,H,D", [
    ([(1, 16, 16), (3, 10, 13)], 3, 128),            # 256 (2 full tiles), 390 (3 tiles + 6-row tail)
    ([(2, 16, 20), (1, 5, 7), (5, 9, 11)], 4, 128),  # 640, 35 (< 1 tile), 495
    ([(4, 16, 16), (1, 1, 1), (1, 3, 43)], 2, 64),   # 1024, L=1 degenerate, 129 (one row into tile 2)
    ([(1, 1, 1)], 1, 128),                           # a single token: O = V, dV = dO, dQ = dK = 0
    ([(3, 16, 16)] + [(1, 2, 3)] * 20, 2, 128),      # one long + many very short sequences
])
def test_multi_tile_ragged_full(orc, grids, H, D):
    w, _, _ = _full_case(orc, inputs.pack(grids, H, D, index=1))
    print(grids, w)


def test_gamma_and_other_rope_split(orc):
    st = inputs.pack([(2, 9, 11), (3, 8, 8)], 2, 128, index=2, rope_dims=(16, 56, 56))
    w, _, _ = _full_case(orc, st, gamma=True)
    print(w)


def test_debug_flags_and_scale(orc):
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(2, 9, 11), (1, 8, 8)], 2, 64, index=2)
    _full_case(orc, st, flags=binding.FLAG_NO_ROPE, oracle_kw=dict(no_rope=True))
    # no_norm: logits are no longer bounded by QK-norm (|s| up to ~30 here): exercises the online-softmax
    # rescaling path; bf16-P error grows with the logit range, gates still hold
    st2 = inputs.pack([(2, 9, 11), (1, 8, 8)], 2, 64, index=2)
    t = inputs.make_inputs(st2, device="cuda")
    t = {k: (v.float() * (0.5 if k in ("q", "k") else 1.0)).to(torch.bfloat16) for k, v in t.items()}
    got = pu.run_gpu(st2, t, flags=binding.FLAG_NO_NORM)
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st2["cu_seqlens"], st2["grids"], dO=a["dO"], no_norm=True)
    pu.check_full(st2, got, ref)
    # explicit softmax scale 0.2 = 1.6 x the default 1/sqrt(64): tau = 1.6, outside the envelope the gates are claimed for
    # (arachne_attn.h "Verified envelope", R19) -> the plan is refused without FLAG_WIDE_LOGITS ...
    with pytest.raises(binding.ArachneError) as ei:
        binding.plan_for(st2, softmax_scale=0.2)
    assert ei.value.status == binding.ERR_LOGIT_RANGE
    # ... and with it, O and all gradients are held to north_star's gates (LSE: test_envelope_lse_* below)
    got = pu.run_gpu(st2, t, flags=binding.FLAG_WIDE_LOGITS, plan_kw=dict(softmax_scale=0.2))
    ref = orc.attention(a["q"], a["k"], a["v"], st2["cu_seqlens"], st2["grids"], dO=a["dO"], scale=0.2)
    print("scale 0.2:", pu.check_full(st2, got, ref, lse=False))


def _large_gamma_case(orc, flags):
    st = inputs.pack([(5, 16, 16)], 2, 128, index=3)
    t = inputs.make_inputs(st, device="cuda")
    g = np.full(128, 3.0, np.float32)
    got = pu.run_gpu(st, t, flags=flags, gamma_q=g, gamma_k=g)
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], gamma_q=g, gamma_k=g)
    return st, got, ref


def test_large_gamma_rescale_path(orc):
    """gamma = 3 on both sides -> tau = 9, logits up to sqrt(D)*9 = 102 (81x the softmax temperature of the BASELINE
    configs): attention is nearly one-hot, the running max grows by more than 2^8 across tiles, so the online-softmax path
    with lazy O-rescale must fire and be right.  O and every gradient are held to north_star's gates, unchanged: the
    backward recomputes S from the forward's fp16 operand images, so P = exp2(S - LSE) stays consistent however large
    the logits are.  (LSE itself is outside the verified envelope here: test_envelope_lse_gamma3_is_bounded_as_documented.)"""
    from paper_2607_01701_b200 import binding
    st, got, ref = _large_gamma_case(orc, binding.FLAG_WIDE_LOGITS)
    w = pu.check_full(st, got, ref, lse=False)
    print("gamma=3:", w)
    # rigorous operand-rounding bound on a logit, hence on LSE: 2^-10 * beta, beta = scale * D * 9 (arachne_attn.h)
    assert w["LSE_abs"] <= 2.0 ** -10 * np.sqrt(128.0) * 9.0
    assert got["plan"].logit_status() == (0, 0.0)                # the flag was set: nothing is recorded


def test_envelope_status_is_raised_without_the_flag(orc):
    """The same gamma = 3 call WITHOUT FLAG_WIDE_LOGITS still runs (gamma is device data) but the plan records that it
    left the envelope: arachne_plan_logit_status -> ARACHNE_ERR_LOGIT_RANGE with tau = 9."""
    from paper_2607_01701_b200 import binding
    st, got, ref = _large_gamma_case(orc, 0)
    pu.check_full(st, got, ref, lse=False)
    status, tau = got["plan"].logit_status()
    assert status == binding.ERR_LOGIT_RANGE and abs(tau - 9.0) < 1e-2, (status, tau)
    # gamma = 1: inside, nothing recorded
    st1 = inputs.structure("tiny")
    got1 = pu.run_gpu(st1, inputs.make_inputs(st1, device="cuda"))
    assert got1["plan"].logit_status() == (0, 0.0)


# Outside the verified envelope (tau > 1) north_star's LSE gate of 1e-3 is NOT claimed (arachne_attn.h "Verified envelope",
# DESIGN.md R19).  What IS claimed there, and therefore tested as a pass / fail statement rather than left as an expected
# failure: the rigorous operand-rounding bound |LSE error| <= 2^-10 * beta, beta = softmax_scale * D * |gamma_q|inf * |gamma_k|inf,
# and the ceiling the header quotes from measurement.  If the forward ever gets a compensated S for wide logits, the
# `> TOL` half of the first test fails and the header's paragraph has to be rewritten.
def test_envelope_lse_gamma3_is_bounded_as_documented(orc):
    from paper_2607_01701_b200 import binding
    st, got, ref = _large_gamma_case(orc, binding.FLAG_WIDE_LOGITS)              # gamma_q = gamma_k = 3: tau = 9
    err = float(np.max(np.abs(pu.to_np(got["LSE"]) - ref["LSE"])))
    beta = (1.0 / np.sqrt(128.0)) * 128.0 * 9.0
    print("LSE max-abs at tau = 9:", err, "bound", 2.0 ** -10 * beta)
    assert err <= 2.0 ** -10 * beta                                               # rigorous
    assert err <= 1.5e-2                                                          # header: "9e-3 at tau = 9" (measured 9.6e-3)
    assert err > pu.TOL["LSE_abs"], "LSE now meets 1e-3 at tau = 9: update the 'Verified envelope' text and this test"


def test_envelope_lse_scale_0p2_is_bounded_as_documented(orc):
    from paper_2607_01701_b200 import binding
    st2 = inputs.pack([(2, 9, 11), (1, 8, 8)], 2, 64, index=2)
    t = inputs.make_inputs(st2, device="cuda")
    t = {k: (v.float() * (0.5 if k in ("q", "k") else 1.0)).to(torch.bfloat16) for k, v in t.items()}
    got = pu.run_gpu(st2, t, flags=binding.FLAG_WIDE_LOGITS, plan_kw=dict(softmax_scale=0.2), with_bwd=False)   # tau = 1.6
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st2["cu_seqlens"], st2["grids"], scale=0.2)
    err = float(np.max(np.abs(pu.to_np(got["LSE"]) - ref["LSE"])))
    print("LSE max-abs at tau = 1.6:", err, "bound", 2.0 ** -10 * 0.2 * 64.0)
    assert err <= 2.0 ** -10 * 0.2 * 64.0                                         # rigorous: 1.25e-2
    assert err <= 2.0e-3                                                          # header: "5e-4..1.2e-3 at tau = 1.6" (at the edge of 1e-3)


# ------------------------------------------------------------------ block-diagonality on the GPU path
def test_poison_neighbours_and_permutation():
    st = inputs.pack([(1, 10, 13), (2, 9, 11), (1, 16, 16)], 2, 128, index=1)   # 130, 198, 256
    cu = st["cu_seqlens"]
    t = inputs.make_inputs(st, device="cuda")
    base = pu.run_gpu(st, t)
    p = {k: v.clone() for k, v in t.items()}
    for k in p:
        p[k][: cu[1]] = 3.0e4            # large finite values in the neighbours (not NaN: 0*NaN would poison a correct mask)
        p[k][cu[2]:] = -3.0e4
    pois = pu.run_gpu(st, p)
    for k in ("O", "dQ", "dK", "dV"):
        assert torch.equal(pois[k][cu[1]:cu[2]], base[k][cu[1]:cu[2]]), k
    assert torch.equal(pois["LSE"][:, cu[1]:cu[2]], base["LSE"][:, cu[1]:cu[2]])
    # packed == the sequence alone (B = 1): bitwise, the schedule is order-preserving per tile
    one = inputs.pack([st["grids"][1]], 2, 128, index=1)
    t1 = {k: v[cu[1]:cu[2]].contiguous() for k, v in t.items()}
    alone = pu.run_gpu(one, t1)
    for k in ("O", "dQ", "dK", "dV"):
        assert torch.equal(alone[k], base[k][cu[1]:cu[2]]), k
    # permuting the sequences permutes the outputs
    perm = torch.cat([torch.arange(cu[2], cu[3]), torch.arange(cu[0], cu[1]), torch.arange(cu[1], cu[2])]).cuda()
    st_p = inputs.pack([st["grids"][2], st["grids"][0], st["grids"][1]], 2, 128, index=1)
    got_p = pu.run_gpu(st_p, {k: v[perm].contiguous() for k, v in t.items()})
    for k in ("O", "dQ", "dK", "dV"):
        assert torch.equal(got_p[k], base[k][perm]), k


@pytest.mark.parametrize("name", ["bucket256", "mixed480p", "cogvideox"])
def test_backward_is_deterministic(name):
    """ARACHNE_FLAG_DETERMINISTIC: bit-identical run to run — the fused kernel reduces its dq~ partial tiles as int32 fixed
    point (integer addition is associative, so the order in which the CTAs' reductions reach L2 cannot matter).  Six runs
    each (an earlier ordered-fp32 scheme differed in one element in one run of ten at the cogvideox shape); the result
    must not depend on what the workspace held."""
    from paper_2607_01701_b200 import binding
    st = inputs.structure(name)
    t = inputs.make_inputs(st, device="cuda")
    plan = binding.plan_for(st, flags=binding.FLAG_DETERMINISTIC)
    ws = torch.empty(plan.workspace_bytes(True), dtype=torch.uint8, device="cuda")
    o, lse = binding.forward(plan, t["q"], t["k"], t["v"])
    runs = []
    for i in range(6):
        ws.fill_(0xA5 if i % 2 == 0 else 0x00)
        runs.append(binding.backward(plan, t["q"], t["k"], t["v"], o, lse, t["dO"], workspace=ws))
        torch.cuda.synchronize()
    for r in runs[1:]:
        for a, b, k in zip(runs[0], r, ("dQ", "dK", "dV")):
            assert torch.equal(a, b), k
    d = binding.backward(binding.plan_for(st), t["q"], t["k"], t["v"], o, lse, t["dO"])     # default (arrival-order) mode
    for a, b in zip(runs[0], d):
        assert float(torch.linalg.vector_norm(a.float() - b.float()) / torch.linalg.vector_norm(b.float())) <= 1e-3


@pytest.mark.parametrize("D", [128, 64])
def test_deterministic_backward_keeps_precision_with_heavy_tailed_dO_and_V(orc, D):
    """The deterministic mode's int32 fixed-point dq~ reduction takes its scale PER QUERY ROW from that row's own |dO_i|
    (bwd_fused.cuh), so a token whose upstream gradient is 1000x the others' must cost the ordinary rows nothing — with one
    scale per (sequence, head) group, as in round 2, they were left ~10 bits short and N(0,1) inputs could not show it.  Two
    dO rows x 1000 and one V row x 1000 (the V maximum enters every row's bound: the documented worst case); dQ of the
    ORDINARY rows is held to north_star's gate, to the default fp32 mode's own error, and row by row to ROW_REL of the row's
    own norm.  A NaN in one dO row must come back as NaN in exactly that dQ row (cvt.rni.s32 alone would make it 0)."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(3, 16, 16), (2, 10, 13)], 2, D, index=7)               # 768 + 260 tokens
    t = dict(inputs.make_inputs(st, device="cuda"))
    g = t["dO"].float(); g[5] *= 1000.0; g[800, 1] *= 1000.0; t["dO"] = g.to(torch.bfloat16)
    v = t["v"].float(); v[100, 0] *= 1000.0; t["v"] = v.to(torch.bfloat16)
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], rope_dims=st["rope_dims"])
    ordinary = np.ones(st["cu_seqlens"][-1], bool)
    ordinary[[5, 800]] = False
    err = {}
    for name, flags in (("fp32", 0), ("fixed", binding.FLAG_DETERMINISTIC)):
        got = pu.run_gpu(st, t, flags=flags)
        dq = pu.to_np(got["dQ"])
        d, n = np.linalg.norm(dq - ref["dQ"], axis=-1), np.linalg.norm(ref["dQ"], axis=-1)
        err[name] = dict(ordinary=pu.rel_l2(dq[ordinary], ref["dQ"][ordinary]), outliers=pu.rel_l2(dq[~ordinary], ref["dQ"][~ordinary]),
                         worst_row=float(np.max((d / np.maximum(n, 1e-300))[ordinary])),
                         dK=pu.rel_l2(pu.to_np(got["dK"]), ref["dK"]), dV=pu.rel_l2(pu.to_np(got["dV"]), ref["dV"]))
        e = err[name]
        assert e["ordinary"] <= pu.TOL["dQ_rel"] and e["outliers"] <= pu.TOL["dQ_rel"], (name, e)
        assert e["dK"] <= pu.TOL["dK_rel"] and e["dV"] <= pu.TOL["dV_rel"], (name, e)
        assert e["worst_row"] <= pu.ROW_REL, (name, e)
    print("heavy-tailed dO / V, D =", D, err)
    assert err["fixed"]["ordinary"] <= 1.25 * err["fp32"]["ordinary"], err      # measured: 1.741e-3 vs 1.736e-3 (D = 128)
    g = t["dO"].float(); g[9, 0, 3] = float("nan"); t["dO"] = g.to(torch.bfloat16)
    got = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC)
    bad = torch.isnan(got["dQ"].float()).any(dim=-1)                            # [N, H]
    want = torch.zeros_like(bad); want[9, 0] = True
    assert torch.equal(bad, want), "a NaN upstream gradient must surface as NaN in its own dQ row, and only there"


# ------------------------------------------------------------------ BASELINE.json configs[1..4] at FULL size,
# in the launch configuration bench.py times: sampled rows + masked-dO + invariants
_REF_CACHE = {}


HEAD_GROUP = 6      # heads per oracle call: its masked-dO dK / dV come back as fp64 [N, heads, D] (1.6 GB at 262k tokens x 6 heads)


def _large_config(orc, name, heads, per_seq=64, order="listed", flags=0):
    """SURVEY §8(c)'s sample: per_seq = 64 query rows per sequence x ALL heads (heads=None), the oracle called one group of
    HEAD_GROUP heads at a time so that host memory stays bounded.  flags: 0 = fused backward (default), FLAG_DETERMINISTIC =
    the deterministic mode; the oracle's O / LSE / dQ rows are computed once per (config, order) and serve both (the second
    user skips the masked-dO dK / dV comparison of the groups it finds cached: those two tensors are not kept)."""
    st = inputs.structure(name, order=order)
    t = inputs.make_inputs(st, device="cuda")
    got = pu.run_gpu(st, t, flags=flags)
    rows = inputs.sample_rows(st, per_seq=per_seq, seed=7)
    ridx = torch.as_tensor(rows, device="cuda")
    # masked-dO backward: dK, dV for ALL key rows depend only on the sampled rows (every head)
    dOm = torch.zeros_like(t["dO"])
    dOm[ridx] = t["dO"][ridx]
    from paper_2607_01701_b200 import binding
    dqm, dkm, dvm = binding.backward(got["plan"], t["q"], t["k"], t["v"], got["O"], got["LSE"], dOm)
    torch.cuda.synchronize()
    # oracle on the sampled rows (needs all K, V of each sequence; Q, dO only at the rows)
    all_heads = list(range(st["H"])) if heads is None else list(heads)
    tc = None
    w = {}
    for g0 in range(0, len(all_heads), HEAD_GROUP):
        grp = all_heads[g0:g0 + HEAD_GROUP]
        key = (name, order, per_seq, tuple(grp))
        ref = _REF_CACHE.get(key)
        if ref is None:
            if tc is None:
                tc = {k: v.cpu().float().numpy() for k, v in t.items()}
            ref = orc.attention_rows(tc["q"], tc["k"], tc["v"], st["cu_seqlens"], st["grids"], rows, dO=tc["dO"], heads=grp,
                                     rope_dims=st["rope_dims"])
            for k_, v_ in pu.check_masked_kv(st, {"dK": dkm, "dV": dvm}, ref).items():
                w[k_] = max(w.get(k_, 0.0), v_)
            _REF_CACHE[key] = {k_: v_ for k_, v_ in ref.items() if k_ not in ("dK", "dV")}
        for k_, v_ in pu.check_rows(st, got, ref, rows).items():
            w[k_] = max(w.get(k_, 0.0), v_)
        del ref
    del tc
    w["rows_x_heads"] = (len(rows), len(all_heads))
    # linearity of the backward in dO (GPU): bwd(dOm) + bwd(dO - dOm) == bwd(dO) within bf16 rounding
    rest = (t["dO"].float() - dOm.float()).to(torch.bfloat16)
    dqr, dkr, dvr = binding.backward(got["plan"], t["q"], t["k"], t["v"], got["O"], got["LSE"], rest)
    for full, m_, r_ in ((got["dK"], dkm, dkr), (got["dV"], dvm, dvr)):
        num = torch.linalg.vector_norm(full.float() - m_.float() - r_.float())
        assert float(num / torch.linalg.vector_norm(full.float())) <= 2e-2
    # full-size invariants on the GPU output
    cu = st["cu_seqlens"]
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        lhs, rhs = got["dV"][s:e].float().sum(0), t["dO"][s:e].float().sum(0)       # sum_j dV_j = sum_i dO_i
        assert float(torch.linalg.vector_norm(lhs - rhs) / torch.linalg.vector_norm(rhs)) <= 2e-2, b
    radial = (got["dQ"].float() * t["q"].float()).sum(-1)                            # RMSNorm: dQ . Q ~ 0
    scale = torch.linalg.vector_norm(got["dQ"].float(), dim=-1) * torch.linalg.vector_norm(t["q"].float(), dim=-1)
    assert float((radial.abs() / scale.clamp_min(1e-20)).mean()) <= 1e-2
    L = torch.as_tensor(np.repeat(np.diff(cu), np.diff(cu)), device="cuda").float()
    assert float((got["LSE"] - L.log()[None]).abs().max()) <= np.sqrt(st["D"]) + 1e-3   # QK-norm bound on LSE
    print(name, order, w)
    return st, t, got


def test_config1_bucket256_sampled_rows_all_heads(orc):
    _large_config(orc, "bucket256", heads=None)


def test_config1_bucket256_reversed_order(orc):
    _large_config(orc, "bucket256", heads=[0, 13, 23], order="reversed")


def test_config2_mixed480p(orc):
    _large_config(orc, "mixed480p", heads=None, per_seq=64, order="shuffled")


def test_config3_long720p(orc):
    st, t, got = _large_config(orc, "long720p", heads=None, per_seq=64)
    # V == 1  =>  O == 1 at full size (softmax normalisation; bf16 rounding of P only)
    from paper_2607_01701_b200 import binding
    ones = torch.ones_like(t["v"])
    o1, _ = binding.forward(got["plan"], t["q"], t["k"], ones)
    assert float((o1.float() - 1.0).abs().max()) <= 1e-2


def test_config4_heavytail(orc):
    _large_config(orc, "heavytail", heads=None, per_seq=64)


# ------------------------------------------------------------------ the deterministic backward at FULL size against the oracle
# (sampled rows + masked-dO + invariants, the same harness and the same oracle rows as the fused default above)
def test_config2_mixed480p_deterministic(orc):
    from paper_2607_01701_b200 import binding
    _large_config(orc, "mixed480p", heads=None, per_seq=64, order="shuffled", flags=binding.FLAG_DETERMINISTIC)


def test_config3_long720p_deterministic(orc):
    from paper_2607_01701_b200 import binding
    _large_config(orc, "long720p", heads=None, per_seq=64, flags=binding.FLAG_DETERMINISTIC)


# ------------------------------------------------------------------ BASELINE.json configs[1] IN FULL, element by element
# ("GPU-vs-oracle on the tiny and 256^2 configs in full"): every O, LSE, dQ, dK, dV element of all 4 sequences x
# 24 heads against orc.attention (3.46 TFLOP-equivalent of plain fp64 loops: about a minute on the GPU box's host cores),
# for the fused backward AND the deterministic one, with the per-row bound of parity_util on top of the per-sequence gates.
def test_config1_bucket256_in_full_fused_and_deterministic(orc):
    from paper_2607_01701_b200 import binding
    st = inputs.structure("bucket256")
    t = inputs.make_inputs(st, device="cuda")
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], rope_dims=st["rope_dims"])
    for name, flags in (("fused", 0), ("deterministic", binding.FLAG_DETERMINISTIC)):
        got = pu.run_gpu(st, t, flags=flags)
        print("bucket256 in full,", name, pu.check_full(st, got, ref))


# ------------------------------------------------------------------ one plan, two streams, two workspaces
def test_one_plan_serves_two_streams_with_separate_workspaces():
    """Every per-launch mutable word (dynamic work counters, logit bound, dS scaling tables) lives in the caller's workspace
    (arachne_attn.h), so two calls on ONE plan that overlap on different streams must both be right."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(4, 16, 16), (9, 16, 16), (3, 10, 13)], 8, 128, index=5)
    t1 = inputs.make_inputs(st, device="cuda")
    t2 = {k: v.flip(0).contiguous() for k, v in t1.items()}          # different bytes on the second stream
    plan = binding.plan_for(st)
    ref = []
    for t in (t1, t2):                                                # one after the other on the current stream
        o, lse = binding.forward(plan, t["q"], t["k"], t["v"])
        ref.append((o, lse) + tuple(binding.backward(plan, t["q"], t["k"], t["v"], o, lse, t["dO"])))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    nb = max(plan.workspace_bytes(False), plan.workspace_bytes(True))
    ws = [torch.empty(nb, dtype=torch.uint8, device="cuda") for _ in range(2)]
    outs = []
    for t in (t1, t2):
        outs.append(dict(o=torch.empty_like(t["q"]), lse=torch.empty((plan.H, plan.N), dtype=torch.float32, device="cuda"),
                         dq=torch.empty_like(t["q"]), dk=torch.empty_like(t["q"]), dv=torch.empty_like(t["q"])))
    for rep in range(3):
        for i, t in enumerate((t1, t2)):                              # interleaved launches, concurrent on the device
            binding.arachne_varlen_attn_fwd(plan, t["q"], t["k"], t["v"], outs[i]["o"], outs[i]["lse"], ws[i], stream=streams[i])
        for i, t in enumerate((t1, t2)):
            binding.arachne_varlen_attn_bwd(plan, t["q"], t["k"], t["v"], outs[i]["o"], outs[i]["lse"], t["dO"], outs[i]["dq"],
                                            outs[i]["dk"], outs[i]["dv"], ws[i], stream=streams[i])
    torch.cuda.synchronize()
    for i in range(2):
        assert torch.equal(outs[i]["o"], ref[i][0]) and torch.equal(outs[i]["lse"], ref[i][1]), i
        assert torch.equal(outs[i]["dv"], ref[i][4]), i                # dV, dK: one owner per tile -> bitwise
        assert torch.equal(outs[i]["dk"], ref[i][3]), i
        num = torch.linalg.vector_norm(outs[i]["dq"].float() - ref[i][2].float())
        assert float(num / torch.linalg.vector_norm(ref[i][2].float())) <= 1e-3, i   # dQ: L2 reduce order is free


# ------------------------------------------------------------------ the CTA-pair (cta_group::2) forward kernel (opt-in, A/B)
@pytest.mark.parametrize("form", ["pairs", "multicast", "multicast+images"])
def test_forward_cluster_forms_against_oracle_and_default(orc, form):
    """The two cluster forms of the forward (head_dim 128): ARACHNE_FLAG_FWD_CTA_PAIRS (cta_group::2 MMAs over a pair that
    holds half of every K/V tile each) and ARACHNE_FLAG_FWD_MULTICAST (two independent CTAs, every K^/V tile fetched half by
    each and multicast into both; with and without the tensor-map path for V).  Items of up to four query tiles: packs
    with 1, 2, 3, 4 and 5+ query tiles per sequence exercise full clusters, a peer CTA with one real + one phantom tile, and a
    peer CTA with only phantoms; ragged last key tiles exercise the multicast of a partial V tile.  Every output is held to
    the oracle gates, and O / LSE must equal the one-CTA kernel's bit for bit (same per-row arithmetic)."""
    from paper_2607_01701_b200 import binding
    flags = {"pairs": binding.FLAG_FWD_CTA_PAIRS, "multicast": binding.FLAG_FWD_MULTICAST,
             "multicast+images": binding.FLAG_FWD_MULTICAST | binding.FLAG_IMAGE_COPIES}[form]
    for grids, H in (([(1, 10, 10), (1, 16, 16), (3, 10, 13), (2, 16, 16), (5, 11, 13)], 3),      # 100, 256, 390, 512, 715 tokens
                     ([(9, 16, 16), (1, 1, 1), (1, 3, 43)], 2)):                                    # 2304 (18 tiles), 1, 129
        st = inputs.pack(grids, H, 128, index=4)
        w, got, t = _full_case(orc, st, flags=flags)
        base = pu.run_gpu(st, t, with_bwd=False)
        assert torch.equal(got["O"], base["O"]) and torch.equal(got["LSE"], base["LSE"])
        print("fwd", form, grids, w)


# ------------------------------------------------------------------ V / dO by tensor-map TMA (default) vs tile-image copies
@pytest.mark.parametrize("D", [64, 128])
def test_raw_tma_tiles_equal_image_copies(orc, D):
    """Default one-shard plans read V (forward, backward) and dO (backward) tiles from the caller's tensors by tensor-map TMA
    (csrc/rawtile.cuh); ARACHNE_FLAG_IMAGE_COPIES is the round-1 path (the prologue copies them into zero-padded tile images).
    The bytes that reach shared memory must be the same, so every output must be bit-identical (deterministic backward) —
    on tails of 5, 2, 8, 123, 127 and 0 rows (whole tiles), i.e. tails below 8 rows, multiples of 8, and both — and a
    neighbouring sequence full of NaN must not leak into a tail tile.  One case is also held to the oracle."""
    from paper_2607_01701_b200 import binding
    grids = [(1, 1, 5), (1, 10, 13), (1, 8, 17), (1, 3, 41), (1, 16, 16), (1, 15, 17)]     # 5, 130, 136, 123, 256, 255 tokens
    st = inputs.pack(grids, 2, D, index=5)
    t = inputs.make_inputs(st, device="cuda")
    raw = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC)
    img = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC | binding.FLAG_IMAGE_COPIES)
    assert raw["plan"].workspace_bytes(True) < img["plan"].workspace_bytes(True)      # no V / dO images in the workspace
    for k in ("O", "LSE", "dQ", "dK", "dV"):
        assert torch.equal(raw[k], img[k]), k
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], rope_dims=st["rope_dims"])
    pu.check_full(st, raw, ref)
    # NaN in every other sequence's V and dO: the remaining sequences are untouched, bit for bit
    cu = st["cu_seqlens"]
    p = {k: v.clone() for k, v in t.items()}
    for b in (0, 2, 4):
        p["v"][cu[b]:cu[b + 1]] = float("nan")
        p["dO"][cu[b]:cu[b + 1]] = float("nan")
    pois = pu.run_gpu(st, p, flags=binding.FLAG_DETERMINISTIC)
    for b in (1, 3, 5):
        for k in ("O", "dQ", "dK", "dV"):
            assert torch.equal(pois[k][cu[b]:cu[b + 1]], raw[k][cu[b]:cu[b + 1]]), (k, b)
        assert torch.equal(pois["LSE"][:, cu[b]:cu[b + 1]], raw["LSE"][:, cu[b]:cu[b + 1]]), b


def test_token_strided_qkv_views_of_a_fused_projection():
    """arachne_attn_params::q_stride / k_stride / v_stride: Q, K, V as the three [:, i] slices of one fused
    [N, 3, H, D] projection output, no .contiguous() — bit-identical to the same data in dense tensors (deterministic
    backward), for both head dims; a stride the plan cannot take is refused."""
    from paper_2607_01701_b200 import binding
    for D in (64, 128):
        st = inputs.pack([(1, 10, 13), (2, 9, 11), (1, 3, 41)], 3, D, index=6)
        t = inputs.make_inputs(st, device="cuda")
        fused = torch.stack([t["q"], t["k"], t["v"]], dim=1).contiguous()            # [N, 3, H, D]
        views = dict(q=fused[:, 0], k=fused[:, 1], v=fused[:, 2], dO=t["dO"])
        assert not views["q"].is_contiguous()
        s3 = 3 * st["H"] * D
        dense = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC)
        strided = pu.run_gpu(st, views, flags=binding.FLAG_DETERMINISTIC, plan_kw=dict(q_stride=s3, k_stride=s3, v_stride=s3))
        for k in ("O", "LSE", "dQ", "dK", "dV"):
            assert torch.equal(dense[k], strided[k]), (D, k)
            assert strided[k].is_contiguous()
        with pytest.raises(TypeError):                                               # undeclared stride: refused by the binding
            pu.run_gpu(st, views, with_bwd=False)
        for bad in (s3 + 4, st["H"] * D - 8):                                         # not a multiple of 8 / overlapping rows
            with pytest.raises(binding.ArachneError) as ei:
                binding.plan_for(st, q_stride=bad)
            assert ei.value.status == 12


@pytest.mark.parametrize("D", [64, 128])
def test_forward_fused_q_equals_prologue(orc, D):
    """ARACHNE_FLAG_FWD_FUSED_Q (the in-kernel variant of §8 a1, SURVEY §7.2 "measure both"): fwd_kernel loads its RAW query
    tiles and applies RMSNorm + 3D RoPE + scale to them itself.  It runs the prologue's arithmetic in the prologue's order
    (csrc/normrope.cuh), so O and LSE must equal the default path's bit for bit — ragged tails (5, 130, 136, 123, 256, 255
    tokens), gamma != 1, and a joint sequence with un-rotated text tokens — and meet the oracle gates."""
    from paper_2607_01701_b200 import binding
    grids = [(1, 1, 5), (1, 10, 13), (1, 8, 17), (1, 3, 41), (1, 16, 16), (1, 15, 17)]
    st = inputs.pack(grids, 2, D, index=7, text_lens=[0, 3, 0, 20, 0, 1])
    t = inputs.make_inputs(st, device="cuda")
    rng = np.random.default_rng(7)
    gq = (1.0 + 0.25 * rng.standard_normal(D)).astype(np.float32)
    gk = (1.0 + 0.25 * rng.standard_normal(D)).astype(np.float32)
    base = pu.run_gpu(st, t, gamma_q=gq, gamma_k=gk, with_bwd=False, flags=binding.FLAG_WIDE_LOGITS)
    fused = pu.run_gpu(st, t, gamma_q=gq, gamma_k=gk, with_bwd=False, flags=binding.FLAG_WIDE_LOGITS | binding.FLAG_FWD_FUSED_Q)
    assert fused["plan"].workspace_bytes(False) == base["plan"].workspace_bytes(False)
    assert torch.equal(fused["O"], base["O"]) and torch.equal(fused["LSE"], base["LSE"])
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], rope_dims=st["rope_dims"], gamma_q=gq, gamma_k=gk,
                        text_lens=st["text_lens"])
    pu.check_full(st, fused, ref, with_bwd=False, lse=False)


def test_forward_backward_capture_into_a_cuda_graph():
    """The calls allocate nothing, synchronise nothing and keep all per-launch state in the caller's workspace, so a forward +
    backward can be captured into a CUDA graph once and replayed (a DiT cascade runs ~60 layers x (2 fwd + 1 bwd) on the same
    packing).  Replays on NEW input values in the same buffers must equal eager calls bit for bit
    (deterministic backward); the tensor maps of V / dO are kernel parameters baked into the graph, which is what fixed
    buffers mean."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(1, 10, 13), (2, 16, 16), (1, 3, 41)], 3, 128, index=8)
    plan = binding.plan_for(st, flags=binding.FLAG_DETERMINISTIC)
    t = inputs.make_inputs(st, device="cuda")
    buf = {k: v.clone() for k, v in t.items()}
    o = torch.empty_like(buf["q"]); lse = torch.empty((plan.H, plan.N), dtype=torch.float32, device="cuda")
    dq, dk, dv = (torch.empty_like(buf["q"]) for _ in range(3))
    ws = torch.empty(max(plan.workspace_bytes(False), plan.workspace_bytes(True)), dtype=torch.uint8, device="cuda")

    def step():
        binding.arachne_varlen_attn_fwd(plan, buf["q"], buf["k"], buf["v"], o, lse, ws)
        binding.arachne_varlen_attn_bwd(plan, buf["q"], buf["k"], buf["v"], o, lse, buf["dO"], dq, dk, dv, ws)

    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        step()                                   # warm-up outside the capture (function attributes are set at plan creation)
    side.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        step()
    for seed in (1, 2):
        new = {k: inputs.randn_bf16(tuple(v.shape), 4242 + 10 * seed + i, v.device) for i, (k, v) in enumerate(t.items())}
        for k in buf:
            buf[k].copy_(new[k])
        g.replay()
        torch.cuda.synchronize()
        got = [x.clone() for x in (o, lse, dq, dk, dv)]
        ref = pu.run_gpu(st, new, flags=binding.FLAG_DETERMINISTIC)
        for a, k in zip(got, ("O", "LSE", "dQ", "dK", "dV")):
            assert torch.equal(a, ref[k]), (seed, k)


@pytest.mark.parametrize("D", [64, 128])
def test_run_to_run_reproducibility_of_everything_but_default_dq(D):
    """A race between warp roles, proxies or CTAs shows up as run-to-run bit differences long before it breaks a tolerance.
    O, LSE, dK, dV have one owner per output tile and must be bit-identical from run to run in EVERY mode, dQ in the deterministic
    mode; 25 runs of a ragged pack (tails of 5, 2, 8, 123, 127 rows, an 18-tile sequence) per kernel form, the workspace
    filled with a different byte before every run."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(1, 1, 5), (1, 10, 13), (1, 8, 17), (1, 3, 41), (1, 16, 16), (1, 15, 17), (9, 16, 16)], 3, D, index=5)
    t = inputs.make_inputs(st, device="cuda")
    forms = [0, binding.FLAG_DETERMINISTIC, binding.FLAG_FWD_FUSED_Q, binding.FLAG_IMAGE_COPIES | binding.FLAG_DETERMINISTIC]
    if D == 128:
        forms += [binding.FLAG_FWD_MULTICAST, binding.FLAG_FWD_CTA_PAIRS]
    for flags in forms:
        plan = binding.plan_for(st, flags=flags)
        ws = torch.empty(max(plan.workspace_bytes(True), plan.workspace_bytes(False)), dtype=torch.uint8, device="cuda")
        ref = None
        for run in range(25):
            ws.fill_(run * 37 % 256)
            o, lse = binding.forward(plan, t["q"], t["k"], t["v"], workspace=ws)
            dq, dk, dv = binding.backward(plan, t["q"], t["k"], t["v"], o, lse, t["dO"], workspace=ws)
            torch.cuda.synchronize()
            cur = dict(O=o, LSE=lse, dK=dk, dV=dv)
            if flags & binding.FLAG_DETERMINISTIC:
                cur["dQ"] = dq
            if ref is None:
                ref = {k: v.clone() for k, v in cur.items()}
                continue
            for k, v in cur.items():
                assert torch.equal(v, ref[k]), (flags, run, k)
        plan.close()
