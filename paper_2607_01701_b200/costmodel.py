"""DiT latency model of the paper, Eq. (9), fitted from THIS kernel's measured times
(first half: the coefficients; the list scheduler + genetic algorithm of Alg. 1 that consume
them are csrc/cascade_sched.cpp, include/arachne_sched.h, bound by scheduler.py).

    L_DiT(B, S, k) = (alpha1 * B*S + alpha2 * B*S^2) / k + V_comm / BW_eff(k)

For the attention of one DiT layer on one GPU (k = 1, no communication) the model reduces to
    t(S) = alpha1 * S + alpha2 * S^2          per sequence (B = 1),
alpha2 capturing "the O(S^2) complexity of the self-attention mechanism" and alpha1 the work linear in the tokens —
here the fused RMSNorm + RoPE prologue, the D = rowsum(dO*O) pass and the un-RoPE / RMSNorm-backward epilogue.
`fit_alpha` is an ordinary least-squares fit through the origin; `sweep` measures fwd+bwd of single sequences of
increasing length through the C ABI with CUDA events.  Host arithmetic only; no attention math lives here.

    python -m paper_2607_01701_b200.costmodel            # on a B200: sweep + fit, prints a markdown table + JSON
"""
from __future__ import annotations

import json
from typing import Sequence, Tuple


def fit_alpha(S: Sequence[float], t: Sequence[float]) -> Tuple[float, float]:
    """Least-squares (alpha1, alpha2) of t = alpha1*S + alpha2*S^2 (Eq. 9 with B = 1, k = 1), weighted by 1/t so that
    short sequences count as much as long ones (relative error)."""
    import numpy as np

    S = np.asarray(S, dtype=np.float64)
    t = np.asarray(t, dtype=np.float64)
    if S.shape != t.shape or S.size < 2:
        raise ValueError("need at least two (S, t) points")
    A = np.stack([S, S * S], axis=1) / t[:, None]
    sol, *_ = np.linalg.lstsq(A, np.ones_like(t), rcond=None)
    return float(sol[0]), float(sol[1])


def predict(alpha1: float, alpha2: float, B: float, S: float, k: int = 1, v_comm: float = 0.0, bw_eff: float = 1.0) -> float:
    """Eq. (9)."""
    return (alpha1 * B * S + alpha2 * B * S * S) / k + v_comm / bw_eff


def sweep(frames=(1, 3, 5, 9, 13, 17, 25, 33), hg=45, wg=80, H=24, D=128, steps=5, warmup=3):
    """fwd+bwd milliseconds of ONE 720p sequence of T latent frames (S = T*45*80 tokens), T in `frames`."""
    import torch

    from . import binding, inputs

    out = []
    for T in frames:
        st = inputs.pack([(T, hg, wg)], H, D, index=3)
        t = inputs.make_inputs(st, device="cuda")
        plan = binding.plan_for(st)
        ws = torch.empty(max(plan.workspace_bytes(False), plan.workspace_bytes(True)), dtype=torch.uint8, device="cuda")
        o = torch.empty_like(t["q"]); lse = torch.empty((H, st["N"]), dtype=torch.float32, device="cuda")
        dq, dk, dv = (torch.empty_like(t["q"]) for _ in range(3))

        def step():
            binding.arachne_varlen_attn_fwd(plan, t["q"], t["k"], t["v"], o, lse, ws)
            binding.arachne_varlen_attn_bwd(plan, t["q"], t["k"], t["v"], o, lse, t["dO"], dq, dk, dv, ws)

        for _ in range(warmup):
            step()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            step()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        out.append(dict(T=T, S=st["N"], ms=ms, tflops=inputs.attention_flops(st) / ms / 1e9))
        plan.close()
        del t, ws, o, lse, dq, dk, dv
    return out


def main():
    pts = sweep()
    a1, a2 = fit_alpha([p["S"] for p in pts], [p["ms"] for p in pts])
    print("| T | S | measured ms | Eq. 9 fit ms | rel. err | TFLOP/s |\n|---|---|---|---|---|---|")
    for p in pts:
        f = predict(a1, a2, 1, p["S"])
        print(f"| {p['T']} | {p['S']} | {p['ms']:.3f} | {f:.3f} | {(f - p['ms']) / p['ms']:+.1%} | {p['tflops']:.0f} |")
    print(json.dumps(dict(alpha1_ms_per_token=a1, alpha2_ms_per_token2=a2, H=24, D=128, points=pts)))


if __name__ == "__main__":
    main()
