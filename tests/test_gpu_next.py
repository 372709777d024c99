"""GPU parity for the SURVEY §8(f) rows built after the base path: NEXT-1 (gamma != 1 with dgamma_q /
dgamma_k outputs, reading R22) and NEXT-2 (joint video + text sequences, reading R21; CogVideoX shape
30 heads x head_dim 64).  Same bar as test_gpu_parity.py: CUDA path through the C ABI vs the
fp64 oracle on the same seeded bytes, north_star's tolerances per tensor and per sequence."""
import numpy as np
import pytest
import torch

from paper_2607_01701_b200 import inputs

import parity_util as pu

pytestmark = pytest.mark.gpu


def _np(t):
    return {k: v.float().cpu().numpy().astype(np.float64) for k, v in t.items()}


def _gammas(D, seed=5):
    rng = np.random.default_rng(seed)
    return (0.5 + rng.random(D)).astype(np.float32), (0.5 + rng.random(D)).astype(np.float32)


def _full(orc, st, flags=0, gamma=True, oracle_kw=None):
    t = inputs.make_inputs(st, device="cuda")
    gq, gk = _gammas(st["D"]) if gamma else (None, None)
    got = pu.run_gpu(st, t, flags=flags, gamma_q=gq, gamma_k=gk, with_dgamma=True)
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], gamma_q=gq, gamma_k=gk,
                        rope_dims=st["rope_dims"], text_lens=st["text_lens"], **(oracle_kw or {}))
    w = pu.check_full(st, got, ref)
    w.update(pu.check_dgamma(got, ref))
    return w, got, t, ref


@pytest.mark.parametrize("grids,text,H,D", [
    ([(2, 9, 11), (1, 8, 8), (1, 1, 1)], [37, 0, 200], 2, 128),    # 235 (text crosses a tile edge), 64, 201
    ([(1, 16, 16), (3, 10, 13)], [128, 6], 3, 64),                 # text = exactly one tile; text fills the tail
    ([(1, 2, 3)] * 5, [1, 0, 250, 3, 0], 2, 128),                  # tiny grids, mostly-text sequences
])
def test_joint_text_tokens_and_dgamma_full(orc, grids, text, H, D):
    w, _, _, _ = _full(orc, inputs.pack(grids, H, D, index=5, text_lens=text))
    print(grids, text, w)


def test_dgamma_video_only_and_deterministic_mode(orc):
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(2, 16, 20), (1, 5, 7), (5, 9, 11)], 4, 128, index=1)
    w, got, t, ref = _full(orc, st)
    print(w)
    # the deterministic (int32 fixed-point reduction) backward feeds the same post kernel: same dgamma gate, and bit-reproducible
    gq, gk = _gammas(128)
    a = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC, gamma_q=gq, gamma_k=gk, with_dgamma=True)
    b = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC, gamma_q=gq, gamma_k=gk, with_dgamma=True)
    pu.check_dgamma(a, ref)
    for k in ("dQ", "dK", "dV", "dGq", "dGk"):
        assert torch.equal(a[k], b[k]), k
    # gamma = None (ones) through the dgamma entry point: dgamma is still defined (d/dgamma at gamma = 1)
    g1 = pu.run_gpu(st, t, with_dgamma=True)
    aa = _np(t)
    r1 = orc.attention(aa["q"], aa["k"], aa["v"], st["cu_seqlens"], st["grids"], dO=aa["dO"], rope_dims=st["rope_dims"])
    pu.check_dgamma(g1, r1)
    # either output may be NULL
    ws = torch.empty(got["plan"].workspace_bytes(True), dtype=torch.uint8, device="cuda")
    dq, dk, dv = (torch.empty_like(t["q"]) for _ in range(3))
    only_k = torch.full((128,), float("nan"), device="cuda")
    binding.arachne_varlen_attn_bwd_dgamma(g1["plan"], t["q"], t["k"], t["v"], g1["O"], g1["LSE"], t["dO"], dq, dk, dv,
                                           None, only_k, ws)
    torch.cuda.synchronize()
    assert torch.equal(only_k, g1["dGk"]) or pu.rel_l2(pu.to_np(only_k), pu.to_np(g1["dGk"])) <= 1e-3


def test_dgamma_is_zero_without_norm(orc):
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(2, 9, 11)], 2, 64, index=2, text_lens=[9])
    t = inputs.make_inputs(st, device="cuda")
    t = {k: (v.float() * (0.5 if k in ("q", "k") else 1.0)).to(torch.bfloat16) for k, v in t.items()}
    got = pu.run_gpu(st, t, flags=binding.FLAG_NO_NORM, with_dgamma=True)
    a = _np(t)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], no_norm=True, text_lens=st["text_lens"])
    pu.check_full(st, got, ref)
    assert not got["dGq"].any() and not got["dGk"].any() and not ref["dGq"].any()


def test_plan_create_joint_validation():
    from paper_2607_01701_b200 import binding
    with pytest.raises(binding.ArachneError) as e:
        binding.Plan([0, 70], [(1, 8, 8)], 2, 64, (16, 24, 24), text_lens=[5])      # 64 + 5 != 70
    assert e.value.status == 5
    with pytest.raises(binding.ArachneError) as e:
        binding.Plan([0, 63], [(1, 8, 8)], 2, 64, (16, 24, 24), text_lens=[-1])
    assert e.value.status == 11
    binding.Plan([0, 70], [(1, 8, 8)], 2, 64, (16, 24, 24), text_lens=[6]).close()


def _large_joint(orc, name, heads=None, per_seq=64, head_group=6):
    """Full-size NEXT-2 workloads in bench.py's launch configuration: SURVEY §8(c)'s sample of 64 query rows per sequence
    (always including text rows) x ALL heads, exact per row; masked-dO dK / dV / dgamma exact for all key rows.  The oracle
    is called one group of `head_group` heads at a time (its dK / dV come back as fp64 [N, heads, D]); dgamma is a sum over
    heads, so each group gets its own GPU backward with dO masked in rows AND heads."""
    from paper_2607_01701_b200 import binding
    st = inputs.structure(name)
    t = inputs.make_inputs(st, device="cuda")
    gq, gk = _gammas(st["D"], seed=9)
    got = pu.run_gpu(st, t, gamma_q=gq, gamma_k=gk, with_dgamma=True)
    cu = st["cu_seqlens"]
    rows = set(inputs.sample_rows(st, per_seq=per_seq, seed=11))
    for b in range(len(cu) - 1):                       # first / middle / last text token of every sequence
        nt = st["text_lens"][b]
        rows.update({cu[b + 1] - nt, cu[b + 1] - nt // 2, cu[b + 1] - 1, cu[b + 1] - nt - 1})
    rows = sorted(rows)
    ridx = torch.as_tensor(rows, device="cuda")
    tc = {k: v.cpu().float().numpy() for k, v in t.items()}
    g_q = torch.as_tensor(gq, device="cuda"); g_k = torch.as_tensor(gk, device="cuda")
    all_heads = list(range(st["H"])) if heads is None else list(heads)
    w = {}
    for g0 in range(0, len(all_heads), head_group):
        grp = all_heads[g0:g0 + head_group]
        ref = orc.attention_rows(tc["q"], tc["k"], tc["v"], cu, st["grids"], rows, dO=tc["dO"], heads=grp, gamma_q=gq, gamma_k=gk,
                                 rope_dims=st["rope_dims"], text_lens=st["text_lens"])
        wg = pu.check_rows(st, got, ref, rows)
        dOm = torch.zeros_like(t["dO"])
        hidx = torch.as_tensor(grp, device="cuda")
        dOm[ridx[:, None], hidx[None, :]] = t["dO"][ridx[:, None], hidx[None, :]]      # masked in rows AND heads
        dqm, dkm, dvm, dgq, dgk = binding.backward(got["plan"], t["q"], t["k"], t["v"], got["O"], got["LSE"], dOm, g_q, g_k,
                                                   with_dgamma=True)
        torch.cuda.synchronize()
        wg.update(pu.check_masked_kv(st, {"dK": dkm, "dV": dvm}, ref))
        wg.update(pu.check_dgamma({"dGq": dgq, "dGk": dgk}, ref))
        for k_, v_ in wg.items():
            w[k_] = max(w.get(k_, 0.0), v_)
        del ref, dOm, dqm, dkm, dvm
    w["rows_x_heads"] = (len(rows), len(all_heads))
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        lhs, rhs = got["dV"][s:e].float().sum(0), t["dO"][s:e].float().sum(0)
        assert float(torch.linalg.vector_norm(lhs - rhs) / torch.linalg.vector_norm(rhs)) <= 2e-2, b
    print(name, w)


def test_cogvideox_shape_full_size(orc):
    _large_joint(orc, "cogvideox")


def test_joint720p_full_size(orc):
    _large_joint(orc, "joint720p")


def test_guard_bands_no_out_of_bounds_writes(orc):
    """compute-sanitizer is closed on this pool, so out-of-bounds WRITES are looked for directly: every output
    tensor and the workspace sit inside a larger allocation whose margins hold a sentinel; after forward + backward
    (fused and deterministic, with dgamma, ragged tails, text tokens) the margins must be untouched."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(1, 10, 13), (2, 9, 11), (1, 1, 1)], 3, 128, index=4, text_lens=[5, 0, 60])   # 135, 198, 61
    t = inputs.make_inputs(st, device="cuda")
    N, H, D = st["N"], st["H"], st["D"]
    G = 4096                                                   # guard elements on each side

    def guarded(numel, dtype, fill):
        buf = torch.full((numel + 2 * G,), fill, dtype=dtype, device="cuda")
        return buf, buf[G:G + numel]

    for flags in (0, binding.FLAG_DETERMINISTIC):
        plan = binding.plan_for(st, flags=flags)
        bufs = {}
        for name in ("o", "dq", "dk", "dv"):
            bufs[name] = guarded(N * H * D, torch.bfloat16, 3.0)
        bufs["lse"] = guarded(H * N, torch.float32, 3.0)
        bufs["dgq"] = guarded(D, torch.float32, 3.0)
        bufs["dgk"] = guarded(D, torch.float32, 3.0)
        wsb = max(plan.workspace_bytes(False), plan.workspace_bytes(True))
        bufs["ws"] = guarded(wsb, torch.uint8, 0x5A)
        v = {k: b[1] for k, b in bufs.items()}
        o, lse = v["o"].view(N, H, D), v["lse"].view(H, N)
        binding.arachne_varlen_attn_fwd(plan, t["q"], t["k"], t["v"], o, lse, v["ws"])
        binding.arachne_varlen_attn_bwd_dgamma(plan, t["q"], t["k"], t["v"], o, lse, t["dO"], v["dq"].view(N, H, D),
                                               v["dk"].view(N, H, D), v["dv"].view(N, H, D), v["dgq"], v["dgk"], v["ws"])
        torch.cuda.synchronize()
        for name, (buf, view) in bufs.items():
            fill = 0x5A if name == "ws" else 3.0
            assert bool((buf[:G] == fill).all()) and bool((buf[G + view.numel():] == fill).all()), (name, flags)
        # and the guarded run computes the right thing
        a = _np(t)
        ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], rope_dims=st["rope_dims"],
                            text_lens=st["text_lens"])
        got = {"O": o, "LSE": lse, "dQ": v["dq"].view(N, H, D), "dK": v["dk"].view(N, H, D), "dV": v["dv"].view(N, H, D),
               "dGq": v["dgq"], "dGk": v["dgk"]}
        pu.check_full(st, got, ref)
        pu.check_dgamma(got, ref)
        plan.close()


def test_host_entry_points_match_device_calls():
    """arachne_varlen_attn_fwd_host / _fwd_bwd_host (the calls bench.py times as `e2e`: cached device buffers, two
    streams, dO uploaded under the forward, O/LSE downloaded under the backward) against the device-pointer calls:
    bit-identical with the deterministic backward, twice in a row on one plan (buffer reuse), pinned and pageable."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(2, 16, 20), (1, 5, 7), (3, 9, 11)], 3, 128, index=2, text_lens=[0, 9, 0])
    t = inputs.make_inputs(st, device="cuda")
    gq, gk = _gammas(128, seed=2)
    ref = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC, gamma_q=gq, gamma_k=gk)
    plan = binding.plan_for(st, flags=binding.FLAG_DETERMINISTIC)
    hgq, hgk = torch.as_tensor(gq), torch.as_tensor(gk)
    for pinned in (True, False, True):
        h = {k: (v.cpu().pin_memory() if pinned else v.cpu()) for k, v in t.items()}
        out = {k: torch.full_like(h["q"], 5.0) for k in ("o", "dq", "dk", "dv")}
        if pinned:
            out = {k: v.pin_memory() for k, v in out.items()}
        lse = torch.zeros((plan.H, plan.N), dtype=torch.float32)
        binding.arachne_varlen_attn_fwd_host(plan, h["q"], h["k"], h["v"], out["o"], lse, hgq, hgk)
        assert torch.equal(out["o"], ref["O"].cpu()) and torch.equal(lse, ref["LSE"].cpu())
        out["o"].fill_(5.0); lse.zero_()
        binding.arachne_varlen_attn_fwd_bwd_host(plan, h["q"], h["k"], h["v"], h["dO"], out["o"], lse, out["dq"], out["dk"],
                                                 out["dv"], hgq, hgk)
        assert torch.equal(out["o"], ref["O"].cpu()) and torch.equal(lse, ref["LSE"].cpu())
        for a, b in (("dq", "dQ"), ("dk", "dK"), ("dv", "dV")):
            assert torch.equal(out[a], ref[b].cpu()), a
    plan.close()


@pytest.mark.parametrize("seed", range(12))
def test_random_packings(orc, seed):
    """Seeded random packings (sequence count, grids, text lengths, heads, head_dim, RoPE split, gamma, backward mode,
    sequence order): every output element by element against the oracle.  Lengths are drawn around tile edges
    (1 .. ~700 tokens) so that single-row tails, exact multiples of 128 and sub-tile sequences all occur."""
    from paper_2607_01701_b200 import binding
    rng = np.random.default_rng(1000 + seed)
    D = int(rng.choice([64, 128]))
    H = int(rng.integers(1, 6))
    B = int(rng.integers(1, 7))
    grids, text = [], []
    for _ in range(B):
        kind = rng.integers(0, 4)
        if kind == 0:
            g = (1, 1, int(rng.integers(1, 130)))
        elif kind == 1:
            g = (int(rng.integers(1, 4)), 8, 16)                       # multiples of 128
        else:
            g = (int(rng.integers(1, 5)), int(rng.integers(1, 14)), int(rng.integers(1, 14)))
        grids.append(g)
        text.append(int(rng.choice([0, 0, 1, 7, 77, 128])))
    half = D // 2
    a = 2 * int(rng.integers(0, half // 2 + 1)); b = 2 * int(rng.integers(0, (D - a) // 4 + 1))
    rope = (a, b, D - a - b)
    st = inputs.pack(grids, H, D, index=7, rope_dims=rope, text_lens=text, order=str(rng.choice(["listed", "reversed", "shuffled"])),
                     seed=seed)
    t = inputs.make_inputs(st, device="cuda")
    gq = (0.5 + rng.random(D)).astype(np.float32)
    gk = (0.5 + rng.random(D)).astype(np.float32)
    flags = binding.FLAG_DETERMINISTIC if rng.integers(0, 2) else 0
    got = pu.run_gpu(st, t, flags=flags, gamma_q=gq, gamma_k=gk, with_dgamma=True)
    x = _np(t)
    ref = orc.attention(x["q"], x["k"], x["v"], st["cu_seqlens"], st["grids"], dO=x["dO"], gamma_q=gq, gamma_k=gk,
                        rope_dims=rope, text_lens=st["text_lens"])
    w = pu.check_full(st, got, ref)
    w.update(pu.check_dgamma(got, ref))
    print(seed, D, H, st["grids"], st["text_lens"], rope, flags, {k: f"{v:.1e}" for k, v in w.items()})
