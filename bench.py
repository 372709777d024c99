#!/usr/bin/env python
"""bench.py — varlen 3D attention fwd+bwd TFLOPS on B200 (BASELINE.json `metric`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload long720p] [--impl reference]

One "step" = one forward + one backward of the whole hot path (prep, fwd, prep, dK/dV, dQ, post
kernels) over one packed batch of synthetic N(0,1) bf16 inputs of the named BASELINE.json config.
`value` = 14*D*H*sum(L_b^2) / t (real lengths; norm/RoPE/softmax and the extra recompute GEMMs of
the deterministic two-pass backward count as time, not FLOPs), inputs resident in HBM.  `e2e` is
the same metric through the C-ABI host call (pinned host buffers, H2D + D2H inside the timed
region).  `roofline` is for the dominant kernel, timed live with CUDA events recorded by the
library on the launching stream.  `cpu_baseline` is the fp64 oracle timed on the host cores on a
bounded sample of the same workload (reported, not a target).  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` capture (profiles/r1b_ncu_720p.md); only known for the workload that was captured.
NCU_TRAFFIC = {("long720p", "bwd_main(fused 5-GEMM | det: dKdV pass)"): 52.91e9, ("long720p", "fwd_kernel"): 6.10e9}

METRIC = "varlen 3D attention fwd+bwd TFLOPS"
UNIT = "TFLOP/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(burst=float(p["bf16_tflops"]), sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    hbm=float(p["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    # fallback stated in B200_PROFILING.md
    return dict(burst=1590.0, sustained=1400.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(st, tensors_cpu, budget_rows=6, heads=2):
    """Time the oracle AS IT STANDS on a bounded sample: fwd + bwd (row-subset / masked-dO mode) for a few
    query rows x `heads` heads of the LONGEST sequence.  Returns (tflops_equiv, seconds, description, cores)."""
    import numpy as np
    from oracle import arachne_oracle as orc

    cu = st["cu_seqlens"]
    b = max(range(len(cu) - 1), key=lambda i: cu[i + 1] - cu[i])
    L = cu[b + 1] - cu[b]
    rows = sorted(set(int(cu[b] + x) for x in np.linspace(0, L - 1, budget_rows).astype(int)))
    hs = list(range(min(heads, st["H"])))
    sl = slice(cu[b], cu[b + 1])
    q, k, v, dO = (tensors_cpu[n][sl].float().numpy() for n in ("q", "k", "v", "dO"))
    rows_local = [r - cu[b] for r in rows]
    t0 = time.perf_counter()
    text = None if not st.get("text_lens") else [st["text_lens"][b]]
    orc.attention_rows(q, k, v, [0, L], [st["grids"][b]], rows_local, dO=dO, heads=hs, rope_dims=st["rope_dims"], text_lens=text)
    dt = time.perf_counter() - t0
    flops = 14.0 * st["D"] * len(rows) * L * len(hs)        # same convention, restricted to the sampled rows
    desc = (f"fp64 oracle fwd+bwd on {len(rows)} query rows x {len(hs)} heads of the longest sequence "
            f"(L={L}) of {st['name']}: {dt:.2f} s")
    return flops / dt / 1e12, dt, desc, orc.num_threads()


def run_reference(args):
    """--impl reference: the oracle on the host cores (this tier's reference arm)."""
    import torch
    from paper_2607_01701_b200 import inputs

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    st = inputs.structure(args.workload)
    st["name"] = args.workload
    from oracle import arachne_oracle as orc
    orc.build()
    # a bounded sample per step so that K+W steps finish within minutes
    sub = {n: None for n in ("q", "k", "v", "dO")}
    cu = st["cu_seqlens"]
    b = max(range(len(cu) - 1), key=lambda i: cu[i + 1] - cu[i])
    L = cu[b + 1] - cu[b]
    one = inputs.pack([st["grids"][b]], st["H"], st["D"], index=st["index"], rope_dims=st["rope_dims"],
                      text_lens=None if not st.get("text_lens") else [st["text_lens"][b]])
    one["name"] = args.workload
    t = inputs.make_inputs(one, device="cpu")
    rows = max(4, min(L, int(5.0e7 / L)))          # ~4 s of oracle time per step on 16 host threads (about 1.4e7 row x key / s)
    times, val = [], 0.0
    for i in range(args.warmup + args.steps):
        v_, dt, desc, cores = oracle_sample(one, t, budget_rows=rows, heads=1)
        if i >= args.warmup:
            times.append(dt); val += v_
    val /= max(len(times), 1)
    ms = 1e3 * sum(times) / max(len(times), 1)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": args.workload, "sample": desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="long720p", choices=["tiny", "bucket256", "mixed480p", "long720p", "heavytail", "joint720p", "cogvideox"])
    ap.add_argument("--impl", default="arachne", choices=["arachne", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--order", default="listed", choices=["listed", "reversed", "shuffled"])
    ap.add_argument("--deterministic", action="store_true", help="ARACHNE_FLAG_DETERMINISTIC: two-pass backward, no atomics")
    ap.add_argument("--heads", type=int, default=0, help="override the head count: the per-rank share of a Ulysses group of degree H/heads")
    ap.add_argument("--seed-offset", type=int, default=0, help="heavytail: another batch drawn from the same recipe (R18)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2607_01701_b200 import binding, inputs     # raises if libarachne_attn.so is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # Multi-GPU (§8 e): sequences/batches are independent -> each rank owns one batch of the same
    # structure (weak scaling), no data-path collective; NCCL only for the barrier and the max-time.
    st = inputs.structure(args.workload, order=args.order, seed_offset=args.seed_offset)
    if args.heads:
        st["H"] = args.heads
    st["name"] = args.workload
    st_r = dict(st, index=st["index"])          # same structure on every rank; different bytes per rank
    t = {k: inputs.randn_bf16((st["N"], st["H"], st["D"]), inputs.BASE_SEED + 16 * st["index"] + tid + 1000 * rank, dev)
         for tid, k in ((1, "q"), (2, "k"), (3, "v"), (4, "dO"))}
    t_plan = time.perf_counter()
    plan = binding.plan_for(st_r, flags=binding.FLAG_DETERMINISTIC if args.deterministic else 0)
    plan_ms = 1e3 * (time.perf_counter() - t_plan)      # host: validation, work lists, LPT order, RoPE / token tables, upload (not in the step)
    ws = torch.empty(max(plan.workspace_bytes(False), plan.workspace_bytes(True)), dtype=torch.uint8, device=dev)
    o = torch.empty_like(t["q"]); lse = torch.empty((plan.H, plan.N), dtype=torch.float32, device=dev)
    dq, dk, dv = (torch.empty_like(t["q"]) for _ in range(3))
    flops = inputs.attention_flops(st)
    s2 = flops / (14.0 * st["D"] * st["H"])

    def step():
        binding.arachne_varlen_attn_fwd(plan, t["q"], t["k"], t["v"], o, lse, ws)
        binding.arachne_varlen_attn_bwd(plan, t["q"], t["k"], t["v"], o, lse, t["dO"], dq, dk, dv, ws)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    plan.enable_profiling(True)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = e0.elapsed_time(e1)
    if world > 1:
        tt = torch.tensor([ms_total], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = float(tt.item())
    ms_step = ms_total / args.steps
    value = world * flops / (ms_step * 1e-3) / 1e12
    kt_f, calls_f = plan.kernel_times(False)
    kt_b, calls_b = plan.kernel_times(True)
    plan.enable_profiling(False)
    launches = args.steps * (plan.num_launches(False) + plan.num_launches(True))

    # ---- e2e through the C-ABI host entry point (pinned host buffers; H2D/D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        nb = t["q"].numel() * 2
        hq, hk, hv, hdo = (x.cpu().pin_memory() for x in (t["q"], t["k"], t["v"], t["dO"]))
        ho, hdq, hdk, hdv = (torch.empty_like(hq).pin_memory() for _ in range(4))
        hlse = torch.empty((plan.H, plan.N), dtype=torch.float32).pin_memory()
        del ws
        torch.cuda.empty_cache()
        binding.arachne_varlen_attn_fwd_bwd_host(plan, hq, hk, hv, hdo, ho, hlse, hdq, hdk, hdv)   # warm-up
        barrier()
        n_e2e = 2
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            binding.arachne_varlen_attn_fwd_bwd_host(plan, hq, hk, hv, hdo, ho, hlse, hdq, hdk, hdv)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        if world > 1:
            tt = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        e2e = {"value": world * flops / dt / 1e12, "unit": UNIT, "h2d_bytes_per_step": 4 * nb,
               "d2h_bytes_per_step": 4 * nb + hlse.numel() * 4, "ms_per_step": dt * 1e3,
               "api": "arachne_varlen_attn_fwd_bwd_host (pinned host buffers)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    # ---- roofline of the dominant kernel: dense contraction -> tensor roofline.
    # Algorithmic FLOPs per launch: fwd_kernel 4*D*H*S2 (2 GEMMs); fused backward kernel
    # 10*D*H*S2 (S, dP, dV, dK, dQ — the 5-GEMM backward convention).
    alg = {"fwd_kernel": 4.0, "bwd_main(fused 5-GEMM | det: dKdV pass)": 10.0}
    kernels = [{"name": n, "ms": ms} for n, ms in kt_f + kt_b]
    dom = max(kernels, key=lambda k_: k_["ms"])
    dom_flops = alg.get(dom["name"], 0.0) * st["D"] * st["H"] * s2
    achieved = dom_flops / (dom["ms"] * 1e-3) / 1e12 if dom["ms"] > 0 else 0.0
    roofline = {"bound": "tensor", "kernel": dom["name"], "achieved": achieved, "peak": peaks["sustained"], "unit": "TFLOP/s",
                "frac": achieved / peaks["sustained"], "traffic": NCU_TRAFFIC.get((args.workload, dom["name"])),
                "traffic_unit": "bytes/launch (ncu dram read+write, profiles/r1b_ncu_720p.md)",
                "peak_source": peaks["source"] + ", bf16_tflops_sustained (kernel timed inside a long step)",
                "kernel_ms": {k_["name"]: round(k_["ms"], 4) for k_ in kernels}, "calls": calls_b}

    cpu = None
    if not args.no_cpu_baseline:
        from oracle import arachne_oracle as orc
        orc.build()
        tc = {k: x.cpu() for k, x in t.items()}
        L_max = max(st["cu_seqlens"][i + 1] - st["cu_seqlens"][i] for i in range(len(st["grids"])))
        # ~10-20 s of oracle time: rows x 2 heads x L_max ~ 2e7 query-row x key products
        v_, dt_, desc, cores = oracle_sample(st, tc, budget_rows=max(8, min(L_max, int(8.0e7 / L_max))), heads=2)
        cpu = {"value": v_, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    # per-CTA finish times of the last launch of the two persistent kernels (arachne_plan_cta_times): what the plan's LPT
    # assignment leaves of the sequence-length skew.  max / mean of the CTA end times; 1.0 = perfectly balanced.
    cta_balance = None
    if rank == 0:
        try:
            cta_balance = {}
            for name, is_bwd in (("fwd_kernel", False), ("bwd_fused_kernel", True)):
                if is_bwd and args.deterministic:
                    continue
                _, end_us = plan.cta_times(is_bwd)
                cta_balance[name] = {"ctas": len(end_us), "end_max_us": max(end_us), "end_mean_us": sum(end_us) / len(end_us),
                                     "end_min_us": min(end_us), "max_over_mean": max(end_us) / (sum(end_us) / len(end_us))}
        except Exception as ex:          # never fail the bench line over a diagnostic
            cta_balance = {"error": str(ex)}
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": args.workload, "order": args.order, "seed_offset": args.seed_offset, "plan_create_ms": round(plan_ms, 3), "deterministic_bwd": bool(args.deterministic), "num_seqs": len(st["grids"]), "total_tokens": st["N"],
                   "heads": st["H"], "head_dim": st["D"], "flop_per_step": flops,
                   "l2": "inputs larger than L2 (4 x %.0f MB bf16 tensors + tiled workspace)" % (t["q"].numel() * 2 / 1e6),
                   "pct_of_measured_bf16_burst": 100.0 * value / world / peaks["burst"],
                   "pct_of_measured_bf16_sustained": 100.0 * value / world / peaks["sustained"],
                   "pct_of_nominal_2250": 100.0 * value / world / 2250.0,
                   "fwd_ms": sum(ms for _, ms in kt_f), "bwd_ms": sum(ms for _, ms in kt_b)},
        "cta_balance": cta_balance, "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
