"""GPU parity of the fused-All-to-All Ulysses calls (include/arachne_attn.h:
arachne_plan_create_sharded, arachne_varlen_attn_{fwd,bwd}_sharded) on ONE GPU.

The k token shards are k separate device allocations and the k "ranks" (head ranges) run one after another on the
same stream: the gather / scatter addressing of the kernels is exactly what runs over NVLink peer mappings on k
GPUs, and no kernel ever waits on another rank's kernel.  Results, reassembled from the shards, are compared with
the fp64 oracle (north_star's gates) and, where the arithmetic is order-preserving, bit for bit with the plain
single-tensor call."""
import numpy as np
import pytest
import torch

from paper_2607_01701_b200 import inputs, ulysses

import parity_util as pu

pytestmark = pytest.mark.gpu


def _split(t, starts):
    # separate allocations (clone), deliberately NOT views of one buffer; pad each by a guard row of NaN-free poison
    return [t[a:b].clone() for a, b in zip(starts, starts[1:])]


def _run_sharded(st, t, k, flags=0, gamma=None, starts=None):
    from paper_2607_01701_b200 import binding
    N, H, D = st["N"], st["H"], st["D"]
    starts = starts or ulysses.token_shard_starts(N, k)
    sh = {n: _split(t[n], starts) for n in ("q", "k", "v", "dO")}
    out = {n: [torch.full_like(x, 7.0) for x in sh["q"]] for n in ("o", "dq", "dk", "dv")}
    gq, gk = (None, None) if gamma is None else (torch.as_tensor(g, dtype=torch.float32, device="cuda") for g in gamma)
    lses, dgq_sum, dgk_sum = [], torch.zeros(D, device="cuda", dtype=torch.float64), torch.zeros(D, device="cuda", dtype=torch.float64)
    plans = []
    for r in range(k):
        off, hl = ulysses.head_range(H, r, k)
        plan = binding.Plan(st["cu_seqlens"], st["grids"], hl, D, st["rope_dims"], flags=flags, text_lens=st.get("text_lens"),
                            shard_starts=starts, total_heads=H, head_offset=off)
        plans.append(plan)
        ws = torch.empty(max(plan.workspace_bytes(False), plan.workspace_bytes(True)), dtype=torch.uint8, device="cuda")
        lse = torch.empty((hl, N), dtype=torch.float32, device="cuda")
        binding.arachne_varlen_attn_fwd_sharded(plan, sh["q"], sh["k"], sh["v"], out["o"], lse, ws, gq, gk)
        lses.append(lse)
    for r in range(k):       # backward after ALL forwards: it reads O rows written by this rank's own forward only
        plan = plans[r]
        ws = torch.empty(plan.workspace_bytes(True), dtype=torch.uint8, device="cuda")
        dgq, dgk = torch.empty(D, device="cuda"), torch.empty(D, device="cuda")
        binding.arachne_varlen_attn_bwd_sharded(plan, sh["q"], sh["k"], sh["v"], out["o"], lses[r], sh["dO"], out["dq"],
                                                out["dk"], out["dv"], ws, dgq, dgk, gq, gk)
        dgq_sum += dgq.double(); dgk_sum += dgk.double()
    torch.cuda.synchronize()
    return {"O": torch.cat(out["o"]), "LSE": torch.cat(lses), "dQ": torch.cat(out["dq"]), "dK": torch.cat(out["dk"]),
            "dV": torch.cat(out["dv"]), "dGq": dgq_sum, "dGk": dgk_sum}


@pytest.mark.parametrize("grids,text,H,D,k", [
    ([(2, 9, 11), (1, 8, 8), (3, 10, 13)], None, 6, 128, 3),       # 198 + 64 + 390 tokens, cuts inside sequences
    ([(1, 16, 16), (1, 5, 7)], [40, 3], 4, 64, 2),                 # joint sequences, D = 64
    ([(1, 2, 3)], None, 8, 128, 8),                                # 6 tokens over 8 ranks: empty shards
])
def test_sharded_equals_oracle_and_plain_call(orc, grids, text, H, D, k):
    from paper_2607_01701_b200 import binding
    st = inputs.pack(grids, H, D, index=6, text_lens=text)
    t = inputs.make_inputs(st, device="cuda")
    rng = np.random.default_rng(1)
    gam = ((0.5 + rng.random(D)).astype(np.float32), (0.5 + rng.random(D)).astype(np.float32))
    got = _run_sharded(st, t, k, gamma=gam)
    a = {n: v.float().cpu().numpy().astype(np.float64) for n, v in t.items()}
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], gamma_q=gam[0], gamma_k=gam[1],
                        rope_dims=st["rope_dims"], text_lens=st["text_lens"])
    w = pu.check_full(st, got, ref)
    w.update(pu.check_dgamma(got, ref))
    print(grids, k, w)
    # the forward and the deterministic backward do the same arithmetic per (sequence, head) whatever the sharding
    plain = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC, gamma_q=gam[0], gamma_k=gam[1])
    det = _run_sharded(st, t, k, flags=binding.FLAG_DETERMINISTIC, gamma=gam)
    for key in ("O", "LSE", "dQ", "dK", "dV"):
        assert torch.equal(det[key], plain[key]), key


def test_sharded_uneven_cuts_bucket256_sampled(orc):
    """BASELINE.json configs[1] at full size with SP degree 4 and UNEVEN token cuts (one inside a tile)."""
    st = inputs.structure("bucket256")
    t = inputs.make_inputs(st, device="cuda")
    starts = [0, 1000, 1001, 9000, st["N"]]
    got = _run_sharded(st, t, 4, starts=starts)
    rows = inputs.sample_rows(st, per_seq=16, seed=3)
    tc = {n: v.cpu().float().numpy() for n, v in t.items()}
    heads = [0, 5, 6, 17, 23]                      # heads of all four ranks
    ref = orc.attention_rows(tc["q"], tc["k"], tc["v"], st["cu_seqlens"], st["grids"], rows, dO=tc["dO"], heads=heads,
                             rope_dims=st["rope_dims"])
    print(pu.check_rows(st, got, ref, rows))
    cu = st["cu_seqlens"]
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        lhs, rhs = got["dV"][s:e].float().sum(0), t["dO"][s:e].float().sum(0)
        assert float(torch.linalg.vector_norm(lhs - rhs) / torch.linalg.vector_norm(rhs)) <= 2e-2, b


def test_sharded_validation():
    from paper_2607_01701_b200 import binding
    kw = dict(cu_seqlens=[0, 64], grids=[(1, 8, 8)], num_heads=2, head_dim=64, rope_dims=(16, 24, 24))
    for bad in (dict(shard_starts=[0, 30, 60], total_heads=4), dict(shard_starts=[0, 40, 30, 64], total_heads=4),
                dict(shard_starts=[0, 64], total_heads=3, head_offset=2), dict(shard_starts=list(range(0, 10)) + [64], total_heads=2)):
        with pytest.raises(binding.ArachneError) as e:
            binding.Plan(**kw, **bad)
        assert e.value.status == 13, bad
    plan = binding.Plan(**kw, shard_starts=[0, 32, 64], total_heads=4, head_offset=2)
    x = torch.zeros(64, 4, 64, dtype=torch.bfloat16, device="cuda")
    lse = torch.empty(2, 64, device="cuda"); ws = torch.empty(plan.workspace_bytes(False), dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.ArachneError) as e:       # a sharded plan through the plain entry point
        binding.arachne_varlen_attn_fwd(plan, x, x, x, x, lse, ws)
    assert e.value.status == 13


# ------------------------------------------------------------------ context parallelism (arachne_plan_create_cp)
def _run_cp(st, t, starts, gamma=None, flags=0):
    """k virtual ranks on one GPU: rank r owns the QUERY tokens of shard r (all heads) and reads K, V of every shard."""
    from paper_2607_01701_b200 import binding
    N, H, D = st["N"], st["H"], st["D"]
    k = len(starts) - 1
    sh = {n: _split(t[n], starts) for n in ("q", "k", "v", "dO")}
    out = {n: [torch.full_like(x, 7.0) for x in sh["q"]] for n in ("o", "dq", "dk", "dv")}
    gq, gk = (None, None) if gamma is None else (torch.as_tensor(g, dtype=torch.float32, device="cuda") for g in gamma)
    plans = [binding.Plan(st["cu_seqlens"], st["grids"], H, D, st["rope_dims"], text_lens=st.get("text_lens"),
                          shard_starts=starts, cp_rank=r, flags=flags) for r in range(k)]
    lses, parts_k, parts_v = [], [], []
    dgq_sum = torch.zeros(D, device="cuda", dtype=torch.float64); dgk_sum = torch.zeros_like(dgq_sum)
    for r in range(k):
        ws = torch.empty(plans[r].workspace_bytes(False), dtype=torch.uint8, device="cuda")
        lse = torch.full((H, N), float("nan"), dtype=torch.float32, device="cuda")
        binding.arachne_varlen_attn_fwd_sharded(plans[r], sh["q"], sh["k"], sh["v"], out["o"], lse, ws, gq, gk)
        lses.append(lse)
    for r in range(k):            # step 1 on every rank (partials poisoned first: unwritten rows must never be read)
        ws = torch.empty(plans[r].workspace_bytes(True), dtype=torch.uint8, device="cuda")
        pk = torch.full((N, H, D), float("nan"), dtype=torch.float32, device="cuda"); pv = torch.full_like(pk, float("nan"))
        dgq = torch.empty(D, device="cuda")
        binding.arachne_varlen_attn_bwd_cp_partial(plans[r], sh["q"], sh["k"], sh["v"], out["o"], lses[r], sh["dO"], out["dq"],
                                                   pk, pv, ws, dgq, gq, gk)
        parts_k.append(pk); parts_v.append(pv); dgq_sum += dgq.double()
    for r in range(k):            # (barrier) step 2 on every rank
        ws = torch.empty(plans[r].workspace_bytes(True), dtype=torch.uint8, device="cuda")
        dgk = torch.empty(D, device="cuda")
        binding.arachne_cp_reduce(plans[r], parts_k, parts_v, sh["k"], out["dk"], out["dv"], ws, dgk, gk)
        dgk_sum += dgk.double()
    torch.cuda.synchronize()
    lse = torch.empty((H, N), dtype=torch.float32, device="cuda")
    for r in range(k):
        lse[:, starts[r]:starts[r + 1]] = lses[r][:, starts[r]:starts[r + 1]]
    return {"O": torch.cat(out["o"]), "LSE": lse, "dQ": torch.cat(out["dq"]), "dK": torch.cat(out["dk"]),
            "dV": torch.cat(out["dv"]), "dGq": dgq_sum, "dGk": dgk_sum}


@pytest.mark.parametrize("grids,text,H,D,starts", [
    ([(2, 9, 11), (1, 8, 8), (3, 10, 13)], None, 3, 128, [0, 100, 300, 652]),        # cuts inside tiles and sequences
    ([(1, 16, 16), (1, 5, 7)], [40, 3], 2, 64, [0, 128, 334]),                       # cut on a tile edge; joint; D = 64
    ([(4, 16, 16), (1, 2, 3)], None, 2, 128, [0, 0, 513, 1030, 1030]),               # empty shards; a rank owning 517 rows
])
def test_context_parallel_equals_oracle(orc, grids, text, H, D, starts):
    st = inputs.pack(grids, H, D, index=6, text_lens=text)
    assert starts[-1] == st["N"]
    t = inputs.make_inputs(st, device="cuda")
    rng = np.random.default_rng(4)
    gam = ((0.5 + rng.random(D)).astype(np.float32), (0.5 + rng.random(D)).astype(np.float32))
    got = _run_cp(st, t, starts, gamma=gam)
    a = {n: v.float().cpu().numpy().astype(np.float64) for n, v in t.items()}
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], gamma_q=gam[0], gamma_k=gam[1],
                        rope_dims=st["rope_dims"], text_lens=st["text_lens"])
    w = pu.check_full(st, got, ref)
    w.update(pu.check_dgamma(got, ref))
    print(grids, starts, w)
    # forward rows are computed exactly as in the plain call: bit-identical O and LSE
    plain = pu.run_gpu(st, t, gamma_q=gam[0], gamma_k=gam[1], with_bwd=False)
    assert torch.equal(got["O"], plain["O"]) and torch.equal(got["LSE"], plain["LSE"])


def test_context_parallel_validation():
    from paper_2607_01701_b200 import binding
    kw = dict(cu_seqlens=[0, 64], grids=[(1, 8, 8)], num_heads=2, head_dim=64, rope_dims=(16, 24, 24))
    with pytest.raises(binding.ArachneError) as e:
        binding.Plan(**kw, shard_starts=[0, 32, 64], cp_rank=2)
    assert e.value.status == 13
    binding.Plan(**kw, shard_starts=[0, 32, 64], cp_rank=0, flags=binding.FLAG_DETERMINISTIC).close()      # accepted (test below)
    plan = binding.Plan(**kw, shard_starts=[0, 32, 64], cp_rank=1)
    x = [torch.zeros(32, 2, 64, dtype=torch.bfloat16, device="cuda") for _ in range(2)]
    lse = torch.empty(2, 64, device="cuda"); ws = torch.empty(plan.workspace_bytes(True), dtype=torch.uint8, device="cuda")
    with pytest.raises(binding.ArachneError) as e:       # a CP plan through the Ulysses backward
        binding.arachne_varlen_attn_bwd_sharded(plan, x, x, x, x, lse, x, x, x, x, ws)
    assert e.value.status == 13


@pytest.mark.parametrize("D", [64, 128])
def test_head_range_of_one_unsharded_tensor_uses_the_tensor_map_path(D):
    """One token shard (the whole tensor) but only a HEAD RANGE per call (total_heads > num_heads, head_offset > 0): such a
    plan is one-shard, so V and dO tiles come by tensor-map TMA with the head coordinate offset (rawtile.cuh RawTensor::head0).
    The two head halves together must equal the plain call bit for bit (deterministic backward), ragged tails included."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(1, 10, 13), (1, 3, 41), (2, 16, 16)], 4, D, index=9)       # 130, 123, 512 tokens
    t = inputs.make_inputs(st, device="cuda")
    plain = pu.run_gpu(st, t, flags=binding.FLAG_DETERMINISTIC)
    halves = _run_sharded(st, t, 2, flags=binding.FLAG_DETERMINISTIC, starts=[0, st["N"]])
    for k in ("O", "dQ", "dK", "dV"):
        assert torch.equal(halves[k], plain[k]), k
    assert torch.equal(halves["LSE"], plain["LSE"])


def test_context_parallel_deterministic_mode(orc):
    """ARACHNE_FLAG_DETERMINISTIC on context-parallel plans: dQ through the int32 fixed-point reduction (order-independent), dK / dV
    through the rank-ordered sum of the partials — three runs bit-identical, and inside the oracle gates."""
    from paper_2607_01701_b200 import binding
    st = inputs.pack([(2, 9, 11), (1, 8, 8), (3, 10, 13)], 3, 128, index=6)
    t = inputs.make_inputs(st, device="cuda")
    starts = [0, 100, 300, 652]
    runs = [_run_cp(st, t, starts, flags=binding.FLAG_DETERMINISTIC) for _ in range(3)]
    for r in runs[1:]:
        for k in ("O", "LSE", "dQ", "dK", "dV"):
            assert torch.equal(r[k], runs[0][k]), k
    a = {n: v.float().cpu().numpy().astype(np.float64) for n, v in t.items()}
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], rope_dims=st["rope_dims"])
    pu.check_full(st, runs[0], ref)
