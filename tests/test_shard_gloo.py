"""Multi-rank host logic (SURVEY §8 e) on CPU: world_size-2 `gloo` processes.

The path shards BY SEQUENCE with no data-path collective (block-diagonal attention: sequences are
independent, BASELINE.json north_star).  Each rank takes the sequences partition_sequences() gives
it, evaluates its own packed sub-batch (here with the oracle standing in for the device: this is
a test of the sharding bookkeeping, not of the kernels), and rank 0 reassembles the global result,
which must equal the single-process evaluation of the whole pack bit for bit.  The only collective
is the max-over-ranks of a scalar time.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01701_b200 import inputs, shard


def test_partition_is_a_balanced_cover():
    lengths = [1024, 2304, 4352, 7424, 256, 256, 7950, 14310, 530, 118800, 3600, 3600]
    for world in (1, 2, 3, 4, 8, 16):
        parts = shard.partition_sequences(lengths, world)
        assert len(parts) == world
        flat = sorted(b for p in parts for b in p)
        assert flat == list(range(len(lengths)))                      # every sequence exactly once
        loads = [sum(shard.seq_cost(lengths[b]) for b in p) for p in parts]
        # LPT list-scheduling bound: max load <= mean load + largest single item
        assert max(loads) <= sum(loads) / world + max(shard.seq_cost(x) for x in lengths)
        assert parts == shard.partition_sequences(lengths, world)       # deterministic
    # more ranks than sequences: the extra ranks own nothing
    parts = shard.partition_sequences([5, 7], 4)
    assert sorted(len(p) for p in parts) == [0, 0, 1, 1]
    with pytest.raises(ValueError):
        shard.partition_sequences([1], 0)


def test_heavytail_partition_balance():
    st = inputs.structure("heavytail")
    cu = st["cu_seqlens"]
    lengths = [cu[i + 1] - cu[i] for i in range(len(cu) - 1)]
    parts = shard.partition_sequences(lengths, 2)
    loads = [sum(shard.seq_cost(lengths[b]) for b in p) for p in parts]
    big = max(shard.seq_cost(x) for x in lengths)
    assert max(loads) <= max(big, sum(loads) / 2 + big / 2 + 1)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import arachne_oracle as orc
        orc.build()
        st = inputs.pack([(1, 8, 8), (2, 10, 10), (1, 5, 7), (3, 6, 6), (1, 1, 1)], 2, 64, index=0)
        t = inputs.make_inputs(st)                                   # same bytes on every rank (seeded)
        a = {k: v.float().numpy().astype(np.float64) for k, v in t.items()}
        mine = shard.shard_structure(st, rank, world)
        idx = np.concatenate([np.arange(s, e) for s, e in mine["token_index"]]) if mine["token_index"] else np.zeros(0, int)
        res = orc.attention(a["q"][idx], a["k"][idx], a["v"][idx], mine["cu_seqlens"], mine["grids"], dO=a["dO"][idx],
                            rope_dims=st["rope_dims"])
        gathered = [None] * world
        dist.all_gather_object(gathered, (idx, res))                 # test-only gather; the product path has none
        slowest = shard.max_over_ranks(10.0 + rank)
        assert slowest == 10.0 + world - 1
        if rank == 0:
            full = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], rope_dims=st["rope_dims"])
            seen = np.zeros(st["N"], dtype=int)
            for ridx, r in gathered:
                seen[ridx] += 1
                for key in ("O", "dQ", "dK", "dV"):
                    assert np.array_equal(r[key], full[key][ridx]), key
                assert np.array_equal(r["LSE"], full["LSE"][:, ridx])
            assert np.all(seen == 1)
            open(os.path.join(out_dir, "ok"), "w").write("ok")
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_shard_equals_single_process(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok").read_text() == "ok"
