"""Multi-GPU host logic (SURVEY §8 e): shard a packed batch across ranks BY SEQUENCE.

Block-diagonal attention never mixes sequences (BASELINE.json north_star), so sequences are
independent units: each rank packs the sequences it owns into its own [N_r, H, D] tensors and
calls arachne_varlen_attn_fwd / _bwd on them.  There is NO data-path collective; the only
cross-rank traffic is the barrier and the max-over-ranks time (NCCL on GPUs, gloo in the CPU
tests).  Balancing sum(L_b^2) per rank is the paper's own problem statement (PAPER.md:23, :41
-- the rank holding the 113-frame bucket runs 58.6 s while the 13-frame rank runs 6.0 s);
here it is the classical longest-processing-time-first greedy on the quadratic cost
(Eq. 9, the alpha_2*B*S^2 term).

This module holds no attention arithmetic: integer bookkeeping and one all_reduce(MAX).
"""
from __future__ import annotations

from typing import List, Sequence


def seq_cost(length: int) -> int:
    """Quadratic attention cost of one sequence (Eq. 9: alpha_2 * S^2)."""
    return int(length) * int(length)


def partition_sequences(lengths: Sequence[int], world_size: int) -> List[List[int]]:
    """Deterministic LPT greedy: sequences in decreasing cost order, each to the least-loaded
    rank (ties -> lowest rank; equal costs -> lower sequence index first).  Every rank computes
    the same assignment from the same lengths, so no communication is needed.  Returns, per
    rank, the sequence indices it owns in increasing order (possibly empty when there are fewer
    sequences than ranks)."""
    if world_size <= 0:
        raise ValueError("world_size must be positive")
    order = sorted(range(len(lengths)), key=lambda b: (-seq_cost(lengths[b]), b))
    load = [0] * world_size
    owned: List[List[int]] = [[] for _ in range(world_size)]
    for b in order:
        r = min(range(world_size), key=lambda i: (load[i], i))
        owned[r].append(b)
        load[r] += seq_cost(lengths[b])
    return [sorted(x) for x in owned]


def shard_structure(st: dict, rank: int, world_size: int) -> dict:
    """The packing structure (inputs.pack layout) of rank `rank`'s shard plus `token_index`:
    for each owned sequence the [start, stop) token range inside the GLOBAL pack, so the caller
    can slice its rows out of global tensors (or scatter results back)."""
    cu = st["cu_seqlens"]
    lengths = [cu[b + 1] - cu[b] for b in range(len(cu) - 1)]
    mine = partition_sequences(lengths, world_size)[rank]
    grids = [tuple(st["grids"][b]) for b in mine]
    lcu = [0]
    for b in mine:
        lcu.append(lcu[-1] + lengths[b])
    text = st.get("text_lens")
    return dict(grids=grids, cu_seqlens=lcu, H=st["H"], D=st["D"], N=lcu[-1], rope_dims=st["rope_dims"],
                text_lens=[text[b] for b in mine] if text else None, index=st.get("index", -1), seq_ids=mine, token_index=[(cu[b], cu[b + 1]) for b in mine])


def max_over_ranks(value: float, device=None) -> float:
    """max over ranks of a scalar (a device-timed duration): the whole-job time is that of the
    slowest rank.  No-op when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
