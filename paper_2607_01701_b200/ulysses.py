"""Ulysses sequence parallelism with the All-to-All fused into the attention kernels.

PAPER.md:84 — "Ulysses SP partitions along the attention-head dimension ... All-to-All"; the SP degree k of a
DiT cascade is the knob Arachne tunes per cascade.  Textbook Ulysses is
    [N/k, H, D] --All-to-All--> [N, H/k, D] --attention--> [N, H/k, D] --All-to-All--> [N/k, H, D]
with two staging tensors and two collectives per pass.  On an NVSwitch domain every GPU can address every peer's
HBM, so here the collectives disappear into the kernels: rank r's `prep_kernel` GATHERS the rows of its H/k heads
straight out of all k token shards (remote loads over NVLink), and the epilogues of `fwd_kernel`,
`bwd_fused_kernel` and `post_kernel` SCATTER O / dV / dQ / dK rows straight into the owners' shards (remote
stores) — tile by tile, overlapped with the tensor-core work of the other CTAs, no staging copy
(include/arachne_attn.h: arachne_plan_create_sharded, arachne_varlen_attn_{fwd,bwd}_sharded).

This module holds NO attention arithmetic: integer bookkeeping (who owns which tokens / heads), the exchange of
peer-mapped buffer addresses, and the barriers that order the ranks.  The bookkeeping is covered by world-size-2
gloo tests on CPU (tests/test_ulysses_gloo.py) and the kernels' gather / scatter by single-GPU tests in which
the k shards are k separate allocations on one device (tests/test_gpu_ulysses.py) — no kernel ever waits on
another rank's kernel.  The drivers below also run as two real processes with real peer mappings (CUDA IPC, both
ranks on the pool's one GPU: tests/test_gpu_multiproc.py); the symmetric-memory transport (`SymmetricShards`) needs k GPUs
(it refuses two ranks on one device) and is the one piece not exercised here.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def token_shard_starts(total_tokens: int, world_size: int) -> List[int]:
    """Token range of each SP rank: the packed batch cut into `world_size` contiguous, near-equal pieces
    (sequences may straddle a cut — positions are looked up through the GLOBAL cu_seqlens).  Returns [k+1]."""
    if world_size <= 0 or total_tokens < 0:
        raise ValueError("world_size must be positive and total_tokens non-negative")
    return [(total_tokens * r) // world_size for r in range(world_size + 1)]


def head_range(total_heads: int, rank: int, world_size: int) -> Tuple[int, int]:
    """(head_offset, local_heads) of a rank.  Ulysses needs the heads to divide evenly (H = 24 -> k in 1,2,3,4,6,8;
    H = 30 (CogVideoX) -> 1,2,3,5,6)."""
    if total_heads % world_size:
        raise ValueError(f"Ulysses needs num_heads ({total_heads}) divisible by the SP degree ({world_size})")
    hl = total_heads // world_size
    return rank * hl, hl


def owner_of_token(starts: Sequence[int], tok: int) -> int:
    """Shard that holds global token `tok` (the rule the kernels use: the LAST r with starts[r] <= tok)."""
    r = 0
    for i in range(1, len(starts) - 1):
        if tok >= starts[i]:
            r = i
    return r


def all_to_all_volume_bytes(total_tokens: int, total_heads: int, head_dim: int, world_size: int, backward: bool) -> int:
    """Bytes ONE rank moves over NVLink per pass: it reads (k-1)/k of its heads' Q,K,V (+ O, dO in backward) rows and
    writes (k-1)/k of its O (dQ, dK, dV) rows; bf16."""
    per_tensor = total_tokens * (total_heads // world_size) * head_dim * 2 * (world_size - 1) // world_size
    return per_tensor * ((5 + 3) if backward else (3 + 1))


def plan_for_rank(st: dict, rank: int, world_size: int, flags: int = 0, **kw):
    """The sharded plan of one SP rank for the packing structure `st` (inputs.pack layout, GLOBAL)."""
    from . import binding

    off, hl = head_range(st["H"], rank, world_size)
    return binding.Plan(st["cu_seqlens"], st["grids"], hl, st["D"], st["rope_dims"], flags=flags,
                        text_lens=st.get("text_lens"), shard_starts=token_shard_starts(st["N"], world_size),
                        total_heads=st["H"], head_offset=off, **kw)


class SymmetricShards:
    """One logical [N, H, D] bf16 tensor sharded by token range over the ranks of `group`, each shard allocated in
    symmetric memory so that every rank holds a device address for every shard (torch.distributed._symmetric_memory:
    CUDA VMM handles exchanged at rendezvous, mapped over NVLink / NVSwitch).  `.local` is this rank's shard (a
    normal torch tensor the rest of the model reads / writes); `.ptrs` is the list the *_sharded calls take."""

    def __init__(self, n_local_max: int, total_heads: int, head_dim: int, group, device):
        import torch
        import torch.distributed._symmetric_memory as symm_mem

        # every rank must allocate the same size: the largest shard
        self.local_full = symm_mem.empty((n_local_max, total_heads, head_dim), dtype=torch.bfloat16, device=device)
        self.handle = symm_mem.rendezvous(self.local_full, group=group)
        self.ptrs = [int(p) for p in self.handle.buffer_ptrs]

    def local(self, n_local: int):
        return self.local_full[:n_local]


class IpcShards:
    """Same interface as SymmetricShards over CUDA IPC (arachne_ipc_alloc / _open): every rank cudaMallocs its shard,
    the 64-byte handles travel through the process group (all_gather_object), every rank maps the others' shards.  Works
    with any backend that can gather python objects (gloo, nccl) and also when several ranks share one GPU — which is how
    the multi-process test runs on a one-GPU box."""

    def __init__(self, n_local_max: int, total_heads: int, head_dim: int, group, device, dtype=None, shape=None):
        import torch
        import torch.distributed as dist

        from . import binding

        self._binding = binding
        self.dtype = dtype or torch.bfloat16
        self.shape = tuple(shape) if shape is not None else (n_local_max, total_heads, head_dim)
        numel = 1
        for x in self.shape:
            numel *= int(x)
        nbytes = max(numel, 1) * torch.empty((), dtype=self.dtype).element_size()
        self._addr, handle = binding.ipc_alloc(nbytes)
        rank, world = dist.get_rank(group), dist.get_world_size(group)
        handles = [None] * world
        dist.all_gather_object(handles, handle, group=group)
        self._opened = []
        self.ptrs = []
        for r in range(world):
            if r == rank:
                self.ptrs.append(self._addr)
            else:
                a = binding.ipc_open(handles[r])
                self._opened.append(a)
                self.ptrs.append(a)
        self.local_full = binding.tensor_from_address(self._addr, self.shape, self.dtype)
        self._group = group

    def local(self, n_local: int):
        return self.local_full[:n_local]

    def close(self):
        import torch
        import torch.distributed as dist

        torch.cuda.synchronize()
        dist.barrier(self._group)                       # nobody is still reading a peer shard
        for a in self._opened:
            self._binding.ipc_close(a)
        self._opened = []
        dist.barrier(self._group)                       # every peer has unmapped before the owner frees
        if self._addr:
            self.local_full = None
            self._binding.ipc_free(self._addr)
            self._addr = 0


class RankSync:
    """Orders the ranks of an SP / CP group around a kernel that reads or writes peer memory.

    Two modes (constructor argument `mode`, else the environment variable ARACHNE_SP_BARRIER, else "host"):

    "host" (default): host synchronisation of the current stream — this rank's kernels, remote stores included, have
    completed — then a host-visible barrier of the group.  Correct by construction on any backend; it is the only mode
    that has ever executed (gloo, in the CPU and one-GPU two-process tests) and therefore the default also under NCCL.

    "stream" (opt-in, NCCL groups only): a one-element all-reduce ENQUEUED ON THE CURRENT STREAM.  It starts after this
    rank's earlier kernels on the stream and finishes only when every rank has entered it, and later kernels on the
    stream start after it — a device-side barrier with no host synchronisation, so the host runs ahead and the launch of
    the next kernel overlaps the wait.  NOT VERIFIED ON HARDWARE: no run on two or more GPUs has taken place (DESIGN.md
    §9), so neither the visibility of the peers' remote stores behind NCCL's kernel nor the ordering has been observed;
    switch it on only together with tests/test_gpu_multiproc.py on a multi-GPU node."""

    MODES = ("host", "stream")

    def __init__(self, group, device, mode=None):
        import os

        import torch
        import torch.distributed as dist

        mode = mode or os.environ.get("ARACHNE_SP_BARRIER", "host")
        if mode not in self.MODES:
            raise ValueError(f"ARACHNE_SP_BARRIER / mode must be one of {self.MODES}, got {mode!r}")
        self._dist, self.group = dist, group
        self.nccl = dist.get_backend(group) == "nccl"
        if mode == "stream" and not self.nccl:
            raise ValueError("the stream-ordered barrier needs an NCCL group (gloo has no device collective)")
        self.on_stream = mode == "stream"
        self.mode = mode
        self._flag = torch.zeros(1, dtype=torch.float32, device=device) if self.on_stream else None

    def describe(self) -> str:
        backend = "NCCL" if self.nccl else "gloo"
        return f"stream-ordered {backend} all-reduce (opt-in, unverified on hardware)" if self.on_stream else f"host sync + {backend} barrier"

    def barrier(self):
        import torch

        if self.on_stream:
            self._dist.all_reduce(self._flag, group=self.group)     # stream-ordered; the host does not wait
        else:
            torch.cuda.current_stream().synchronize()               # my kernels (incl. their remote stores) have completed
            self._dist.barrier(self.group)

    def all_reduce_sum(self, t):
        """Sum a small device tensor over the group (dgamma partials: 2 x D floats)."""
        if self.nccl:
            self._dist.all_reduce(t, group=self.group)              # an ordinary device collective on the tensor's own data
            return t
        host = t.cpu()
        self._dist.all_reduce(host, group=self.group)
        return host.to(t.device)


class UlyssesAttention:
    """Forward / backward of the packed attention over an SP group of k GPUs in one NVSwitch domain.

    Each rank owns the tokens [starts[r], starts[r+1]) of the pack (all heads) in `self.q/k/v/o/dO/dq/dk/dv.local`
    and computes heads head_range(H, r, k) for ALL tokens.  forward(): barrier (every rank's Q,K,V are in place) ->
    arachne_varlen_attn_fwd_sharded (gather + attention + scatter) -> barrier (every rank's O shard is complete).
    The barriers are the only collectives on the data path; dgamma partials are all-reduced (2 x D floats)."""

    def __init__(self, st: dict, group=None, flags: int = 0, transport: str = "symm"):
        import torch
        import torch.distributed as dist

        from . import binding

        self.group = group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.st = st
        self.starts = token_shard_starts(st["N"], self.world)
        self.n_local = self.starts[self.rank + 1] - self.starts[self.rank]
        n_max = max(self.starts[r + 1] - self.starts[r] for r in range(self.world))
        dev = torch.device("cuda", torch.cuda.current_device())
        self.plan = plan_for_rank(st, self.rank, self.world, flags=flags)
        names = ("q", "k", "v", "o", "dO", "dq", "dk", "dv")
        Shards = SymmetricShards if transport == "symm" else IpcShards      # "ipc": CUDA IPC (arachne_ipc_*)
        self.buf = {n: Shards(n_max, st["H"], st["D"], group, dev) for n in names}
        self.lse = torch.empty((self.plan.H, st["N"]), dtype=torch.float32, device=dev)
        self.ws = torch.empty(max(self.plan.workspace_bytes(False), self.plan.workspace_bytes(True)), dtype=torch.uint8, device=dev)
        self._binding = binding
        self._dist = dist
        self._sync = RankSync(group, dev)

    def local(self, name: str):
        return self.buf[name].local(self.n_local)

    def _barrier(self):
        self._sync.barrier()

    def forward(self, gamma_q=None, gamma_k=None):
        b = self.buf
        self._barrier()
        self._binding.arachne_varlen_attn_fwd_sharded(self.plan, b["q"].ptrs, b["k"].ptrs, b["v"].ptrs, b["o"].ptrs,
                                                      self.lse, self.ws, gamma_q, gamma_k)
        self._barrier()
        return self.local("o")

    def backward(self, gamma_q=None, gamma_k=None, with_dgamma=False):
        import torch

        b = self.buf
        dgq = dgk = None
        if with_dgamma:
            dgq = torch.empty(self.st["D"], dtype=torch.float32, device=self.lse.device)
            dgk = torch.empty_like(dgq)
        self._barrier()
        self._binding.arachne_varlen_attn_bwd_sharded(self.plan, b["q"].ptrs, b["k"].ptrs, b["v"].ptrs, b["o"].ptrs,
                                                      self.lse, b["dO"].ptrs, b["dq"].ptrs, b["dk"].ptrs, b["dv"].ptrs,
                                                      self.ws, dgq, dgk, gamma_q, gamma_k)
        if with_dgamma:        # gamma is shared by all heads (R1): sum the per-rank partials (2 x D floats)
            both = self._sync.all_reduce_sum(torch.stack([dgq, dgk]))
            dgq, dgk = both[0], both[1]
        self._barrier()
        return self.local("dq"), self.local("dk"), self.local("dv"), dgq, dgk

    def close(self):
        for b in self.buf.values():
            if hasattr(b, "close"):
                b.close()
        self.plan.close()
