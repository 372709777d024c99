"""Ulysses host logic on CPU: world_size-2 `gloo` processes.

What is checked (no kernels here — those are tests/test_gpu_ulysses.py):
  * token_shard_starts / head_range / owner_of_token are a consistent cover on every rank;
  * the GATHER RULE the kernels implement (row (tok - starts[r]) of shard r = owner_of_token(tok), heads
    [head_offset, head_offset + H/k)) delivers exactly the tensor the textbook Ulysses All-to-All delivers, and the
    SCATTER RULE is its inverse (round trip == identity);
  * head-sharded evaluation (the oracle standing in for the device) + all_reduce of the dgamma partials equals the
    single-process evaluation: O, dQ, dK, dV bit for bit per head, LSE per head, dgamma to rounding.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01701_b200 import inputs, ulysses


def test_bookkeeping_is_a_cover():
    for N, k in ((264, 2), (118800, 8), (7, 8), (15104, 3), (1, 1)):
        s = ulysses.token_shard_starts(N, k)
        assert s[0] == 0 and s[-1] == N and len(s) == k + 1 and all(b >= a for a, b in zip(s, s[1:]))
        assert max(b - a for a, b in zip(s, s[1:])) - min(b - a for a, b in zip(s, s[1:])) <= 1
        for tok in {0, N - 1, N // 2, *s[1:-1], *(x - 1 for x in s[1:-1] if x > 0)}:
            r = ulysses.owner_of_token(s, tok)
            assert s[r] <= tok < s[r + 1]
    heads = [ulysses.head_range(24, r, 8) for r in range(8)]
    assert heads == [(3 * r, 3) for r in range(8)]
    with pytest.raises(ValueError):
        ulysses.head_range(30, 0, 4)
    assert ulysses.all_to_all_volume_bytes(118800, 24, 128, 8, False) == 118800 * 3 * 128 * 2 * 7 // 8 * 4


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _gather_rule(shards, starts, off, hl, N):
    """[N, hl, D] as the sharded kernels read it."""
    rows = []
    for tok in range(N):
        r = ulysses.owner_of_token(starts, tok)
        rows.append(shards[r][tok - starts[r], off:off + hl])
    return np.stack(rows)


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import arachne_oracle as orc
        orc.build()
        st = inputs.pack([(1, 8, 8), (2, 5, 7), (1, 1, 1), (1, 6, 6)], 4, 64, index=0, text_lens=[3, 0, 2, 0])
        N, H, D = st["N"], st["H"], st["D"]
        starts = ulysses.token_shard_starts(N, world)
        off, hl = ulysses.head_range(H, rank, world)
        full = {k: v.float().numpy().astype(np.float64) for k, v in inputs.make_inputs(st).items()}
        mine = {k: v[starts[rank]:starts[rank + 1]] for k, v in full.items()}      # what this rank owns: its tokens, all heads
        # --- textbook Ulysses All-to-All #1 (send peer p the heads of p, receive my heads of peer p's tokens)
        recv = {}
        for name in ("q", "k", "v", "dO"):
            send = [torch.from_numpy(np.ascontiguousarray(mine[name][:, ulysses.head_range(H, p, world)[0]:][:, :hl])) for p in range(world)]
            got = [None] * world
            for p in range(world):                  # gloo has no all_to_all: k gathers, one per destination
                lst = [None] * world if rank == p else None
                dist.gather_object(send[p], lst, dst=p)
                if rank == p:
                    got = lst
            recv[name] = np.concatenate([g.numpy() for g in got])              # [N, hl, D] head-sharded
        # --- the kernels' gather rule, applied to all shards (rank-local view of peer memory)
        all_shards = [None] * world
        dist.all_gather_object(all_shards, mine)
        for name in ("q", "k", "v", "dO"):
            via_rule = _gather_rule([s[name] for s in all_shards], starts, off, hl, N)
            assert np.array_equal(via_rule, recv[name]), name
            assert np.array_equal(via_rule, full[name][:, off:off + hl])
        # --- head-sharded evaluation on the GLOBAL packing (sequences straddle the token cut: positions come from cu_seqlens)
        gq, gk = 0.5 + np.arange(D) / D, 1.5 - np.arange(D) / D
        res = orc.attention(recv["q"], recv["k"], recv["v"], st["cu_seqlens"], st["grids"], dO=recv["dO"], gamma_q=gq,
                            gamma_k=gk, rope_dims=st["rope_dims"], text_lens=st["text_lens"])
        dg = torch.from_numpy(np.stack([res["dGq"], res["dGk"]]))
        dist.all_reduce(dg)                                                       # gamma is shared by all heads (R1)
        # --- scatter rule = All-to-All #2: every rank writes its heads of every token into the owner's shard
        out_shards = [None] * world
        dist.all_gather_object(out_shards, {k: res[k] for k in ("O", "dQ", "dK", "dV")})
        mine_out = {k: np.concatenate([out_shards[p][k][starts[rank]:starts[rank + 1]] for p in range(world)], axis=1)
                    for k in ("O", "dQ", "dK", "dV")}                              # [n_r, H, D], heads in rank order
        ref = orc.attention(full["q"], full["k"], full["v"], st["cu_seqlens"], st["grids"], dO=full["dO"], gamma_q=gq,
                            gamma_k=gk, rope_dims=st["rope_dims"], text_lens=st["text_lens"])
        for k in ("O", "dQ", "dK", "dV"):
            assert np.array_equal(mine_out[k], ref[k][starts[rank]:starts[rank + 1]]), k
        assert np.array_equal(res["LSE"], ref["LSE"][off:off + hl])
        assert np.allclose(dg[0].numpy(), ref["dGq"], rtol=1e-12, atol=1e-12)
        assert np.allclose(dg[1].numpy(), ref["dGk"], rtol=1e-12, atol=1e-12)
        open(os.path.join(out_dir, f"ok{rank}"), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_ulysses_rules_equal_all_to_all(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok0").read_text() == "ok" and (tmp_path / "ok1").read_text() == "ok"


def test_context_parallel_bookkeeping():
    from paper_2607_01701_b200 import context_parallel as cp
    cu = [0, 198, 262, 652, 653, 1700]
    N = cu[-1]
    for starts in ([0, 100, 300, 652, N], [0, 0, 513, 1030, N], [0, N], cp.balanced_starts(cu, 3), cp.balanced_starts(cu, 8)):
        assert starts[0] == 0 and starts[-1] == N and all(b >= a for a, b in zip(starts, starts[1:]))
        for b in range(len(cu) - 1):
            s, L = cu[b], cu[b + 1] - cu[b]
            covered = np.zeros((L + 127) // 128, dtype=int)
            for r in range(len(starts) - 1):
                first, n = cp.query_tile_range(s, L, starts[r], starts[r + 1])
                rows = [t for t in range(s, s + L) if starts[r] <= t < starts[r + 1]]              # brute force
                tiles = sorted({(t - s) // 128 for t in rows})
                assert tiles == list(range(first, first + n))
                covered[first:first + n] += 1
                assert (r in cp.contributors(starts, s, L)) == bool(rows)
            assert np.all(covered >= 1)                      # every query tile has an owner (boundary tiles: two)
        costs = [cp.rank_cost(cu, starts[r], starts[r + 1]) for r in range(len(starts) - 1)]
        assert sum(costs) == sum((cu[i + 1] - cu[i]) ** 2 for i in range(len(cu) - 1))
    # cost-balanced cuts: no rank more than one row-of-the-longest-sequence above the mean
    for k in (2, 3, 8):
        st = cp.balanced_starts(cu, k)
        costs = [cp.rank_cost(cu, st[r], st[r + 1]) for r in range(k)]
        assert max(costs) <= sum(costs) / k + max(cu[i + 1] - cu[i] for i in range(len(cu) - 1))


def test_rank_sync_defaults_to_the_host_barrier_and_stream_mode_is_opt_in(tmp_path, monkeypatch):
    """ulysses.RankSync: the stream-ordered NCCL barrier has never run on two GPUs, so it must be asked for
    (mode="stream" / ARACHNE_SP_BARRIER=stream) and is refused on a group that has no device collective."""
    import pytest
    import torch.distributed as dist

    from paper_2607_01701_b200 import ulysses

    monkeypatch.delenv("ARACHNE_SP_BARRIER", raising=False)
    dist.init_process_group("gloo", init_method=f"file://{tmp_path}/rdzv", rank=0, world_size=1)
    try:
        s = ulysses.RankSync(dist.group.WORLD, "cpu")
        assert s.mode == "host" and not s.on_stream and "host sync" in s.describe()
        with pytest.raises(ValueError):
            ulysses.RankSync(dist.group.WORLD, "cpu", mode="stream")          # gloo: no device collective
        with pytest.raises(ValueError):
            ulysses.RankSync(dist.group.WORLD, "cpu", mode="sometimes")
        monkeypatch.setenv("ARACHNE_SP_BARRIER", "stream")
        with pytest.raises(ValueError):
            ulysses.RankSync(dist.group.WORLD, "cpu")                          # the variable is honoured (and refused on gloo)
    finally:
        dist.destroy_process_group()
