"""Context parallelism without a ring ("CP ... K/V ring").

Each rank owns a contiguous token range of the packed batch (all heads) and computes the attention of ITS query tokens
against all keys of their sequences.  Inside one NVSwitch domain the K/V "ring" is unnecessary: the kernels read the
other ranks' K and V rows straight from their shards (peer memory), and the reduce-scatter of dK / dV is the owner
reading the other ranks' fp32 partials in rank order (include/arachne_attn.h: arachne_plan_create_cp,
arachne_varlen_attn_bwd_cp_partial, arachne_cp_reduce).  Unlike Ulysses the degree is not tied to the head count.

This module holds the integer bookkeeping (mirrors of what the plan computes, used by the tests and for sizing) and
the multi-GPU driver; no attention arithmetic.  Verified: kernels on one GPU with k shard buffers
(tests/test_gpu_ulysses.py), bookkeeping on CPU (tests/test_ulysses_gloo.py); not run on k GPUs (one-GPU pool).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

TILE = 128


def query_tile_range(seq_start: int, seq_len: int, lo: int, hi: int) -> Tuple[int, int]:
    """(first tile, tile count) of a sequence's 128-row query tiles that hold tokens of [lo, hi) (global indices)."""
    a, b = max(lo, seq_start), min(hi, seq_start + seq_len)
    if a >= b:
        return 0, 0
    first = (a - seq_start) // TILE
    return first, (b - 1 - seq_start) // TILE + 1 - first


def contributors(starts: Sequence[int], seq_start: int, seq_len: int) -> List[int]:
    """Ranks whose query range intersects the sequence: the ranks whose dK / dV partials its keys must sum."""
    return [r for r in range(len(starts) - 1)
            if starts[r + 1] > starts[r] and starts[r] < seq_start + seq_len and starts[r + 1] > seq_start]


def rank_cost(cu_seqlens: Sequence[int], lo: int, hi: int) -> int:
    """Quadratic cost (query rows x keys) of the rank that owns queries [lo, hi): sum over sequences of rows * L
    (Eq. 9's alpha2 term).  Equal token counts do NOT mean equal cost when lengths differ."""
    c = 0
    for b in range(len(cu_seqlens) - 1):
        s, e = cu_seqlens[b], cu_seqlens[b + 1]
        rows = max(0, min(hi, e) - max(lo, s))
        c += rows * (e - s)
    return c


def balanced_starts(cu_seqlens: Sequence[int], world_size: int) -> List[int]:
    """Token cuts that equalise rank_cost (not token counts): walk the tokens in order, cut when the running cost
    passes r/k of the total.  Cuts may fall inside a sequence."""
    N = cu_seqlens[-1]
    total = rank_cost(cu_seqlens, 0, N)
    starts, acc, r = [0], 0, 1
    for b in range(len(cu_seqlens) - 1):
        s, e = cu_seqlens[b], cu_seqlens[b + 1]
        L = e - s
        while r < world_size and acc + L * L >= total * r / world_size:
            need = total * r / world_size - acc            # cost still missing for cut r, at L per row
            starts.append(min(e, s + int(-(-need // L))))
            r += 1
        acc += L * L
    while len(starts) < world_size:
        starts.append(N)
    return starts + [N]


class ContextParallelAttention:
    """Forward / backward over a CP group of k GPUs in one NVSwitch domain (torch.distributed + symmetric memory).
    forward(): barrier -> fwd_sharded -> barrier (a rank writes only its own O shard, but it READS its peers' Q, K, V
    shards: nobody may overwrite its inputs for the next layer until every rank's kernels are done with them).
    backward(): barrier -> bwd_cp_partial -> barrier -> cp_reduce -> all-reduce of the dgamma parts -> barrier.
    The barriers are ulysses.RankSync's: host barriers by default, stream-ordered under NCCL with ARACHNE_SP_BARRIER=stream."""

    def __init__(self, st: dict, group=None, starts=None, transport: str = "symm"):
        import torch
        import torch.distributed as dist

        from . import binding
        from .ulysses import IpcShards, RankSync, SymmetricShards

        self.group, self._dist, self._binding = group, dist, binding
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.starts = list(starts) if starts is not None else balanced_starts(st["cu_seqlens"], self.world)
        self.n_local = self.starts[self.rank + 1] - self.starts[self.rank]
        n_max = max(self.starts[r + 1] - self.starts[r] for r in range(self.world))
        dev = torch.device("cuda", torch.cuda.current_device())
        self.plan = binding.Plan(st["cu_seqlens"], st["grids"], st["H"], st["D"], st["rope_dims"],
                                 text_lens=st.get("text_lens"), shard_starts=self.starts, cp_rank=self.rank)
        Shards = SymmetricShards if transport == "symm" else IpcShards
        self.buf = {n: Shards(n_max, st["H"], st["D"], group, dev) for n in ("q", "k", "v", "o", "dO", "dq", "dk", "dv")}
        self.part = {}
        for n in ("dk_partial", "dv_partial"):            # fp32 [N,H,D] partial buffers every rank can read
            if transport == "symm":
                import torch.distributed._symmetric_memory as symm_mem
                t = symm_mem.empty((st["N"], st["H"], st["D"]), dtype=torch.float32, device=dev)
                self.part[n] = (t, [int(p) for p in symm_mem.rendezvous(t, group=group).buffer_ptrs], None)
            else:
                sh = IpcShards(0, 0, 0, group, dev, dtype=torch.float32, shape=(st["N"], st["H"], st["D"]))
                self.part[n] = (sh.local_full, sh.ptrs, sh)
        self.lse = torch.empty((st["H"], st["N"]), dtype=torch.float32, device=dev)
        self.ws = torch.empty(max(self.plan.workspace_bytes(False), self.plan.workspace_bytes(True)), dtype=torch.uint8, device=dev)
        self._sync = RankSync(group, dev)
        self._D = st["D"]

    def _barrier(self):
        self._sync.barrier()

    def forward(self, gamma_q=None, gamma_k=None):
        b = self.buf
        self._barrier()
        self._binding.arachne_varlen_attn_fwd_sharded(self.plan, b["q"].ptrs, b["k"].ptrs, b["v"].ptrs, b["o"].ptrs, self.lse,
                                                      self.ws, gamma_q, gamma_k)
        self._barrier()              # every rank has finished READING its peers' Q, K, V before anyone reuses them
        return b["o"].local(self.n_local)

    def backward(self, gamma_q=None, gamma_k=None, with_dgamma=False):
        """-> (dq, dk, dv, dgamma_q, dgamma_k) of this rank's tokens; dgamma (reading R22) is the sum over ALL ranks
        (step 1 yields this rank's part of dgamma_q, step 2 its part of dgamma_k; both are all-reduced), or None."""
        import torch

        b = self.buf
        dgq = dgk = None
        if with_dgamma:
            dgq = torch.empty(self._D, dtype=torch.float32, device=self.lse.device)
            dgk = torch.empty_like(dgq)
        self._barrier()
        self._binding.arachne_varlen_attn_bwd_cp_partial(self.plan, b["q"].ptrs, b["k"].ptrs, b["v"].ptrs, b["o"].ptrs, self.lse,
                                                         b["dO"].ptrs, b["dq"].ptrs, self.part["dk_partial"][0],
                                                         self.part["dv_partial"][0], self.ws, dgq, gamma_q, gamma_k)
        self._barrier()
        self._binding.arachne_cp_reduce(self.plan, self.part["dk_partial"][1], self.part["dv_partial"][1], b["k"].ptrs,
                                        b["dk"].ptrs, b["dv"].ptrs, self.ws, dgk, gamma_k)
        if with_dgamma:
            if self.n_local == 0:                    # a rank without tokens launches no row: its parts are zero
                dgq.zero_(); dgk.zero_()
            both = self._sync.all_reduce_sum(torch.stack([dgq, dgk]))
            dgq, dgk = both[0], both[1]
        self._barrier()
        return b["dq"].local(self.n_local), b["dk"].local(self.n_local), b["dv"].local(self.n_local), dgq, dgk

    def close(self):
        for b in list(self.buf.values()) + [p[2] for p in self.part.values() if p[2] is not None]:
            if hasattr(b, "close"):
                b.close()
        self.plan.close()
