"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no RMSNorm, RoPE, softmax, attention):
only (a) the packing structure of the five BASELINE.json workloads and (b) a counter-based
N(0,1) -> bf16 generator.  Both the CUDA path and the oracle RECEIVE the bytes made here; the
side that did not generate never regenerates.

The workloads stand in for the paper's WebVid / Koala-36M / Lynx batches, which
are not available: shapes follow PAPER.md:41 (13..113-frame buckets), :100 (33K..262K tokens),
:306 (129-frame cap), :312-316 (24 heads x head_dim 128) via BASELINE.json `configs`.
"""
from __future__ import annotations

import math
import torch

BASE_SEED = 260701701          # + 16*config_index + tensor_id  (0 structure, 1 Q, 2 K, 3 V, 4 dO)
CONFIG_NAMES = ["tiny", "bucket256", "mixed480p", "long720p", "heavytail",
                # SURVEY §8(f) NEXT-2 workloads (not BASELINE.json configs): joint video+text sequences
                "joint720p", "cogvideox"]

_M64 = (1 << 64) - 1


def _splitmix64(state: int):
    """One step of SplitMix64 on python ints (structure draws only)."""
    state = (state + 0x9E3779B97F4A7C15) & _M64
    z = state
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return state, z ^ (z >> 31)


def rope_dims_for(D: int):
    """(d_t, d_h, d_w): 16/24/24 for D=64 (BASELINE.json configs[0]); doubled for D=128 (reading R6)."""
    return {64: (16, 24, 24), 128: (32, 48, 48)}[D]


def heavytail_structure(seed: int, max_tokens: int = 262144):
    """Reading R18: resolution uniform over {256x256, 480x848, 720x1280} (latent Hg x Wg = /16),
    latent frames T in {1,4,9,17,29,33} with P(T) ~ 1/T, i.i.d.; a draw that would push N over
    max_tokens is rejected; stop after 64 consecutive rejections."""
    res = [(16, 16), (30, 53), (45, 80)]
    frames = [1, 4, 9, 17, 29, 33]
    w = [1.0 / t for t in frames]
    tot = sum(w)
    cdf, acc = [], 0.0
    for x in w:
        acc += x / tot
        cdf.append(acc)
    state = seed & _M64
    grids, n, rejected = [], 0, 0
    while rejected < 64:
        state, r1 = _splitmix64(state)
        state, r2 = _splitmix64(state)
        hg, wg = res[r1 % 3]
        u = (r2 >> 11) / float(1 << 53)
        t = frames[next(i for i, c in enumerate(cdf) if u <= c or i == len(cdf) - 1)]
        L = t * hg * wg
        if n + L > max_tokens:
            rejected += 1
            continue
        rejected = 0
        grids.append((t, hg, wg))
        n += L
    return grids


def structure(name: str, seed_offset: int = 0, order: str = "listed"):
    """Packing structure of a BASELINE.json config: dict(grids, cu_seqlens, H, D, rope_dims, index).
    order: 'listed' | 'reversed' | 'shuffled' (sequence order inside the pack)."""
    idx = CONFIG_NAMES.index(name)
    text_lens = None
    if name == "tiny":
        grids, H, D = [(1, 8, 8), (2, 10, 10)], 2, 64
    elif name == "bucket256":
        grids, H, D = [(4, 16, 16), (9, 16, 16), (17, 16, 16), (29, 16, 16)], 24, 128
    elif name == "mixed480p":
        grids, H, D = [(5, 30, 53), (9, 30, 53), (17, 30, 53), (33, 30, 53)], 24, 128
    elif name == "long720p":
        grids, H, D = [(33, 45, 80)], 24, 128
    elif name == "heavytail":
        grids, H, D = heavytail_structure(BASE_SEED + 16 * idx + seed_offset), 24, 128
    elif name == "joint720p":
        # the 720p long clip with its text prompt joined to the sequence (HunyuanVideo single-stream blocks,
        # PAPER.md:322; "text ... < 256 tokens"), 24 heads x 128
        grids, H, D, text_lens = [(33, 45, 80)], 24, 128, [256]
    elif name == "cogvideox":
        # CogVideoX-shaped batch: 30 heads x head_dim 64, 4 joint sequences of a 13-frame
        # 30x45 latent grid plus a 226-token prompt each
        grids, H, D, text_lens = [(13, 30, 45)] * 4, 30, 64, [226] * 4
    else:
        raise KeyError(name)
    return pack(grids, H, D, order=order, seed=BASE_SEED + 16 * idx + seed_offset, index=idx, text_lens=text_lens)


def pack(grids, H, D, order="listed", seed=0, index=-1, rope_dims=None, text_lens=None):
    """text_lens [B] (optional): text tokens appended after the video tokens of each sequence (reading R21)."""
    grids = [tuple(int(x) for x in g) for g in grids]
    text = [0] * len(grids) if text_lens is None else [int(x) for x in text_lens]
    assert len(text) == len(grids)
    seqs = list(zip(grids, text))
    if order == "reversed":
        seqs = seqs[::-1]
    elif order == "shuffled":
        state = (seed ^ 0xA5A5A5A5) & _M64
        for i in range(len(seqs) - 1, 0, -1):
            state, r = _splitmix64(state)
            j = r % (i + 1)
            seqs[i], seqs[j] = seqs[j], seqs[i]
    grids, text = [g for g, _ in seqs], [x for _, x in seqs]
    cu = [0]
    for (t, hg, wg), nt in seqs:
        cu.append(cu[-1] + t * hg * wg + nt)
    return dict(grids=grids, cu_seqlens=cu, H=H, D=D, N=cu[-1],
                rope_dims=tuple(rope_dims) if rope_dims else rope_dims_for(D), index=index,
                text_lens=text if any(text) else None)


def attention_flops(st) -> float:
    """FLOP count convention of BASELINE.json `metric`: 4*D*H*sum(L^2) forward, 10*D*H*sum(L^2)
    backward (five LxLxD GEMMs incl. the S recompute); real lengths, not tile-padded."""
    cu = st["cu_seqlens"]
    s2 = sum((cu[i + 1] - cu[i]) ** 2 for i in range(len(cu) - 1))
    return 14.0 * st["D"] * st["H"] * s2


# ------------------------------------------------------------------ counter-based N(0,1) -> bf16
def _i64(x: int) -> int:
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    return (z >> k) & ((1 << (64 - k)) - 1)


def randn_bf16(shape, seed: int, device="cpu", chunk: int = 1 << 24) -> torch.Tensor:
    """Element-addressable N(0,1) rounded RNE to bf16: element i of the flattened tensor is a
    SplitMix64-style mix of (seed, i) -> two 24-bit uniforms -> Box-Muller in fp32 -> bf16.
    Runs on whichever torch device it is given (CPU here, CUDA on the GPU box); the bytes it
    returns are THE input for both the CUDA path and the oracle."""
    numel = 1
    for s in shape:
        numel *= int(s)
    out = torch.empty(numel, dtype=torch.bfloat16, device=device)
    c1, c2, g = _i64(0xBF58476D1CE4E5B9), _i64(0x94D049BB133111EB), _i64(0x9E3779B97F4A7C15)
    s0 = _i64(seed * 0xD1342543DE82EF95 + 0x2545F4914F6CDD1D)
    for start in range(0, numel, chunk):
        n = min(chunk, numel - start)
        z = torch.arange(start + 1, start + 1 + n, dtype=torch.int64, device=device) * g + s0
        z = (z ^ _lsr(z, 30)) * c1
        z = (z ^ _lsr(z, 27)) * c2
        z = z ^ _lsr(z, 31)
        u1 = (_lsr(z, 40).to(torch.float32) + 1.0) * (1.0 / 16777216.0)        # (0, 1]
        u2 = ((z >> 16) & 0xFFFFFF).to(torch.float32) * (1.0 / 16777216.0)     # [0, 1)
        x = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
        out[start:start + n] = x.to(torch.bfloat16)
    return out.view(*shape)


def make_inputs(st, device="cpu", with_dO=True):
    """Q, K, V (and dO) ~ N(0,1) bf16 [N,H,D] for a packing structure `st` (seeds per DESIGN.md §4)."""
    base = BASE_SEED + 16 * max(st.get("index", 0), 0)
    shape = (st["N"], st["H"], st["D"])
    t = {name: randn_bf16(shape, base + tid, device) for tid, name in ((1, "q"), (2, "k"), (3, "v"))}
    if with_dO:
        t["dO"] = randn_bf16(shape, base + 4, device)
    return t


def sample_rows(st, per_seq: int = 64, seed: int = 0):
    """Seeded sample of query rows per sequence (global token indices, sorted): always rows
    0, 127, 128, L-1 and the first row of the tail tile (128*floor((L-1)/128)), plus random rows."""
    cu = st["cu_seqlens"]
    state = (BASE_SEED * 31 + seed) & _M64
    rows = []
    for b in range(len(cu) - 1):
        L = cu[b + 1] - cu[b]
        s = {0, L - 1, min(127, L - 1), min(128, L - 1), 128 * ((L - 1) // 128)}
        while len(s) < min(per_seq, L):
            state, r = _splitmix64(state)
            s.add(r % L)
        rows.extend(cu[b] + x for x in sorted(s))
    return rows


# ------------------------------------------------------------------ synthetic cascade-scheduling instances (NEXT-4)
def cascade_instance(seed: int, n_samples: int = 8, degrees=(1, 2, 4, 8), n_gpus: int = 16):
    """A seeded scheduling instance shaped like one Arachne training batch: per sample a VAE
    cascade followed by a DiT cascade (edge VAE -> DiT), sample lengths from the heavy-tailed recipe (R18).  The
    latency / feasibility TABLES are synthetic numbers with the shape of Eq. 8-9 (work/k + a per-degree overhead; small
    degrees infeasible for long samples) — no cost model of the method is evaluated here.  Returns plain lists."""
    grids = heavytail_structure(BASE_SEED + 977 * seed, max_tokens=1 << 30)[:n_samples]
    state = (seed * 0x9E3779B97F4A7C15 + 12345) & _M64
    K = [int(k) for k in degrees]
    L, feas, preds = [], [], []
    for i, (t, hg, wg) in enumerate(grids):
        S = t * hg * wg
        state, r1 = _splitmix64(state)
        state, r2 = _splitmix64(state)
        jit1, jit2 = 0.9 + 0.2 * ((r1 >> 11) / float(1 << 53)), 0.9 + 0.2 * ((r2 >> 11) / float(1 << 53))
        vae = [jit1 * (2.0e-4 * S) / k + 0.02 * (k - 1) for k in K]                       # VAE: linear in tokens
        dit = [jit2 * (3.0e-4 * S + 2.5e-9 * S * S) * 60 / 1000 / k + 0.05 * math.log2(k) for k in K]   # DiT: Eq. 9 shape
        L.append(vae); feas.append([True] * len(K)); preds.append([])
        L.append(dit); feas.append([S / k <= 70000 for k in K]); preds.append([2 * i])    # activation memory ~ tokens / k
        if not any(feas[-1]):
            feas[-1][-1] = True
    return dict(K=K, L=L, feasible=feas, preds=preds, N=n_gpus)
