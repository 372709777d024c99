#!/usr/bin/env python
"""bench.py — varlen 3D attention fwd+bwd TFLOPS on B200 (BASELINE.json `metric`).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload long720p] [--impl reference] [--sp ulysses|cp]

One "step" = one forward + one backward of the whole hot path (prep, fwd, prep, scale, bwd_fused, post kernels)
over one packed batch of synthetic N(0,1) bf16 inputs of the named BASELINE.json config.
`value` = 14*D*H*sum(L_b^2) / t (real lengths; norm/RoPE/softmax and every prologue / epilogue kernel count as time, not
FLOPs), inputs resident in HBM.  `e2e` is the same metric through the C-ABI host call (pinned host buffers, H2D + D2H
inside the timed region; median of >= 5 repetitions).  `roofline` is for the dominant kernel, timed live with CUDA events
recorded by the library on the launching stream.  `cpu_baseline` is the fp64 oracle timed on the host cores on a bounded
sample of the same workload (reported, not a target).  `config.targets` carries BOTH north_star targets in one record:
the 720p long clip (>= 60 % of the measured bf16 burst peak) and the heavy-tailed batch (>= 50 %), plus the deterministic
backward on the main workload.  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "varlen 3D attention fwd+bwd TFLOPS"
UNIT = "TFLOP/s"
WORKLOADS = ["tiny", "bucket256", "mixed480p", "long720p", "heavytail", "joint720p", "cogvideox"]
TRAFFIC_CSV = os.path.join("profiles", "r3_traffic.csv")      # transcribed from ncu captures (profiles/r3_ncu.md names the commands)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(burst=float(p["bf16_tflops"]), sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    hbm=float(p["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    # fallback stated in B200_PROFILING.md
    return dict(burst=1590.0, sustained=1400.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


def kernel_source_hash() -> str:
    """sha256 over the CUDA sources: ties an ncu capture to the kernels it was taken from."""
    d = os.path.join(ROOT, "paper_2607_01701_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            with open(os.path.join(d, f), "rb") as fh:
                h.update(f.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed captures — only those taken
    from the kernels as they are now (source hash).  The figure moves from launch to launch (what the 126 MB L2 happens to
    keep of the backward's ~122 MB per-head working set), so the CSV holds SEVERAL captures per kernel and this returns
    their median with the spread: (median or None, {"min", "max", "captures", "source"} or the reason)."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None, {"source": f"{TRAFFIC_CSV} absent"}
    vals, stale, reports = [], None, []
    with open(path) as f:
        for row in csv.DictReader(f):
            if row["workload"] == workload and row["kernel"] in kernel:
                if row["src_sha"] != kernel_source_hash():
                    stale = row["src_sha"]
                    continue
                vals.append(float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]))
                if row["report"] not in reports:
                    reports.append(row["report"])
    if not vals:
        why = (f"capture predates the current kernels (src {stale} != {kernel_source_hash()})" if stale
               else f"no row for {workload} / {kernel}")
        return None, {"source": f"{TRAFFIC_CSV}: {why}"}
    vals.sort()
    n = len(vals)
    med = vals[n // 2] if n % 2 else 0.5 * (vals[n // 2 - 1] + vals[n // 2])
    return med, {"min": vals[0], "max": vals[-1], "captures": n, "source": f"{TRAFFIC_CSV} ({'; '.join(reports)}, src {kernel_source_hash()})"}


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


def self_launch_argv(argv, n_gpus, port, python=None):
    """Command line that re-runs this bench as `n_gpus` ranks of ONE node (one process per GPU): the driver's launch contract,
    `python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py <same flags>`.
    Pure function of its arguments (tests/test_bench_launch.py)."""
    return [python or sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(n_gpus)}",
            "--master-addr", "127.0.0.1", "--master-port", str(int(port)), os.path.join(ROOT, "bench.py")] + list(argv)


def needs_self_launch(args, environ) -> bool:
    """`python bench.py --gpus N` (N > 1) outside torchrun: nobody has started the other ranks, so this process must.
    The reference arm never needs ranks (rank 0 alone times the oracle on the host cores)."""
    return args.gpus > 1 and "WORLD_SIZE" not in environ and args.impl != "reference"


def free_port() -> int:
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def self_launch(args, argv) -> int:
    """Start the N ranks and hand their exit code back.  Fails loudly, before anything is launched, when the node has
    fewer than N GPUs: a bench line that says n_gpus = N must have run on N devices."""
    import torch
    have = torch.cuda.device_count() if torch.cuda.is_available() else 0
    if have < args.gpus and (args.sp == "none" or have == 0):
        # (--sp ulysses|cp may run with fewer devices than ranks: sp_bench.py then shares device 0 and says config.emulated)
        raise SystemExit(f"bench.py --gpus {args.gpus}: this node has {have} CUDA device(s); refusing to emulate ranks on fewer GPUs")
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")            # the communicator log shows which transport (NVLS / P2P) each rank got
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    return subprocess.call(self_launch_argv(argv, args.gpus, free_port()), env=env)


def run_reference(args):
    """--impl reference: the oracle on the host cores (this tier's reference arm)."""
    from paper_2607_01701_b200 import inputs

    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    st = inputs.structure(args.workload)
    st["name"] = args.workload
    from oracle import arachne_oracle as orc
    orc.build()
    # a bounded sample per step so that K+W steps finish within minutes
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


class Env:
    """Process-wide context: ranks, device, barrier."""

    def __init__(self):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback")
        if self.local_rank >= torch.cuda.device_count():
            raise SystemExit(f"bench.py: rank {self.rank} has no GPU of its own (LOCAL_RANK {self.local_rank}, "
                             f"{torch.cuda.device_count()} device(s)): one process per GPU, ranks are never stacked on a device")
        torch.cuda.set_device(self.local_rank)
        self.dev = torch.device("cuda", self.local_rank)
        if self.world > 1:
            os.environ.setdefault("NCCL_DEBUG", "INFO")          # (before the communicator exists) transport / NVLS lines of the init
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            dist.init_process_group("nccl", device_id=self.dev)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, x: float) -> float:
        if self.world == 1:
            return x
        tt = self.torch.tensor([x], device=self.dev, dtype=self.torch.float64)
        self.dist.all_reduce(tt, op=self.dist.ReduceOp.MAX)
        return float(tt.item())


def time_workload(env: Env, workload, steps, warmup, deterministic=False, order="listed", seed_offset=0, heads=0, keep=False, extra_flags=0):
    """W untimed + K timed steps of `workload` (device-resident inputs; every rank its own batch of the same structure).
    Returns the measurement dict (and, with keep, the live objects for the e2e / cpu_baseline legs)."""
    torch = env.torch
    from paper_2607_01701_b200 import binding, inputs     # raises if libarachne_attn.so is missing

    st = inputs.structure(workload, order=order, seed_offset=seed_offset)
    if heads:
        st["H"] = heads
    st["name"] = workload
    t = {k: inputs.randn_bf16((st["N"], st["H"], st["D"]), inputs.BASE_SEED + 16 * st["index"] + tid + 1000 * env.rank, env.dev)
         for tid, k in ((1, "q"), (2, "k"), (3, "v"), (4, "dO"))}
    t_plan = time.perf_counter()
    plan = binding.plan_for(st, flags=(binding.FLAG_DETERMINISTIC if deterministic else 0) | extra_flags)
    plan_ms = 1e3 * (time.perf_counter() - t_plan)      # host: validation, work lists, LPT order, RoPE / token tables, upload (not in the step)
    ws = torch.empty(max(plan.workspace_bytes(False), plan.workspace_bytes(True)), dtype=torch.uint8, device=env.dev)
    o = torch.empty_like(t["q"]); lse = torch.empty((plan.H, plan.N), dtype=torch.float32, device=env.dev)
    dq, dk, dv = (torch.empty_like(t["q"]) for _ in range(3))
    flops = inputs.attention_flops(st)

    def step():
        binding.arachne_varlen_attn_fwd(plan, t["q"], t["k"], t["v"], o, lse, ws)
        binding.arachne_varlen_attn_bwd(plan, t["q"], t["k"], t["v"], o, lse, t["dO"], dq, dk, dv, ws)

    warmup = max(warmup, 3)
    for _ in range(warmup):
        step()
    env.barrier()
    plan.enable_profiling(True)
    sampler = ClockSampler(env.local_rank)
    if env.rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    env.barrier()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    env.barrier()
    clocks = sampler.stop() if env.rank == 0 else None
    ms_total = env.max_over_ranks(e0.elapsed_time(e1))
    ms_step = ms_total / steps
    kt_f, _ = plan.kernel_times(False)
    kt_b, calls_b = plan.kernel_times(True)
    plan.enable_profiling(False)
    r = dict(workload=workload, st=st, flops=flops, ms_step=ms_step, ms_total=ms_total, steps=steps, warmup=warmup,
             value=env.world * flops / (ms_step * 1e-3) / 1e12, kt_f=kt_f, kt_b=kt_b, calls_b=calls_b, clocks=clocks,
             plan_ms=plan_ms, launches=steps * (plan.num_launches(False) + plan.num_launches(True)),
             tensor_mb=t["q"].numel() * 2 / 1e6, deterministic=deterministic)
    cta_balance = None
    if env.rank == 0:
        # per-CTA finish times of the last launch of the two persistent kernels (arachne_plan_cta_times): what the plan's LPT
        # order + dynamic hand-out leaves of the sequence-length skew.  max / mean of the CTA end times; 1.0 = balanced.
        try:
            cta_balance = {}
            for name, is_bwd in (("fwd_kernel", False), ("bwd_fused_kernel", True)):
                _, end_us = plan.cta_times(is_bwd)
                cta_balance[name] = {"ctas": len(end_us), "end_max_us": max(end_us), "end_mean_us": sum(end_us) / len(end_us),
                                     "end_min_us": min(end_us), "max_over_mean": max(end_us) / (sum(end_us) / len(end_us))}
        except Exception as ex:          # never fail the bench line over a diagnostic
            cta_balance = {"error": str(ex)}
    r["cta_balance"] = cta_balance
    if keep:
        r.update(plan=plan, t=t, ws=ws)
    else:
        plan.close()
    return r


def roofline_block(r, peaks):
    """`roofline` object of one measurement (time_workload result): the dominant kernel against the tensor roofline.
    Algorithmic FLOPs per launch: fwd_kernel 4*D*H*S2 (2 GEMMs); backward main kernel 10*D*H*S2 (S, dP, dV,
    dK, dQ — the 5-GEMM backward convention), S2 = sum_b L_b^2."""
    st = r["st"]
    s2 = r["flops"] / (14.0 * st["D"] * st["H"])
    alg = {"fwd_kernel": 4.0, "bwd_fused_kernel": 10.0}
    kernels = [{"name": n, "ms": ms} for n, ms in r["kt_f"] + r["kt_b"]]
    dom = max(kernels, key=lambda k_: k_["ms"])
    dom_flops = alg.get(dom["name"], 0.0) * st["D"] * st["H"] * s2
    achieved = dom_flops / (dom["ms"] * 1e-3) / 1e12 if dom["ms"] > 0 else 0.0
    # Denominator (B200_PROFILING.md): the sustained figure for a kernel timed inside a long step, the burst figure for one
    # that runs alone at boost clocks.  Decided by the length of ONE step of the workload — a property of the workload, not of
    # --steps (the loop of warm-up + timed steps is continuous load either way): a step of >= 100 ms keeps the GPU at its 1 kW
    # cap for seconds even at the minimum of 3 + 1 steps.  `frac_of_burst` / `frac_of_sustained` are always both reported;
    # `frac_of_burst` is the one north_star's targets are stated in.
    long_run = r["ms_step"] >= 100.0
    peak_kind = "bf16_tflops_sustained (%.0f ms / step, warm-up + timed steps back to back: power-capped clocks)" % r["ms_step"] if long_run \
        else "bf16_tflops burst (%.2f ms / step: boost clocks)" % r["ms_step"]
    peak = peaks["sustained"] if long_run else peaks["burst"]
    traffic, tinfo = ncu_traffic(r["workload"], dom["name"])
    return {"bound": "tensor", "kernel": dom["name"], "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
            "frac": achieved / peak, "frac_denominator": "sustained" if long_run else "burst", "frac_of_burst": achieved / peaks["burst"],
            "frac_of_sustained": achieved / peaks["sustained"],
            "traffic": traffic, "traffic_unit": "bytes/launch (ncu dram__bytes_read.sum + dram__bytes_write.sum; median of the captures)",
            "traffic_min": tinfo.get("min"), "traffic_max": tinfo.get("max"), "traffic_captures": tinfo.get("captures", 0),
            "traffic_source": tinfo["source"], "peak_source": peaks["source"] + ", " + peak_kind,
            "kernel_ms": {k_["name"]: round(k_["ms"], 4) for k_ in kernels}, "calls": r["calls_b"]}


def target_entry(r, peaks, target_pct=None):
    e = {"tflops": round(r["value"], 1), "ms_per_step": round(r["ms_step"], 3), "steps": r["steps"],
         "pct_of_measured_bf16_burst": round(100.0 * r["value"] / r["world"] / peaks["burst"], 2),
         "sm_mhz": r["clocks"]["sm_mhz"] if r["clocks"] else None, "reasons": r["clocks"]["reasons"] if r["clocks"] else None,
         "fwd_ms": round(sum(ms for _, ms in r["kt_f"]), 3), "bwd_ms": round(sum(ms for _, ms in r["kt_b"]), 3)}
    if target_pct is not None:
        e["north_star_target_pct_of_burst"] = target_pct
        e["met"] = e["pct_of_measured_bf16_burst"] >= target_pct
    return e


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="long720p", choices=WORKLOADS)
    ap.add_argument("--impl", default="arachne", choices=["arachne", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-targets", action="store_true", help="skip the extra legs (heavytail, deterministic) of config.targets")
    ap.add_argument("--order", default="listed", choices=["listed", "reversed", "shuffled"])
    ap.add_argument("--deterministic", action="store_true", help="ARACHNE_FLAG_DETERMINISTIC backward as the main measurement")
    ap.add_argument("--fwd-pairs", action="store_true", help="ARACHNE_FLAG_FWD_CTA_PAIRS: the CTA-pair (cta_group::2) forward kernel (A/B)")
    ap.add_argument("--fwd-mcast", action="store_true", help="ARACHNE_FLAG_FWD_MULTICAST: forward as clusters of 2 sharing the K/V stream by TMA multicast (A/B)")
    ap.add_argument("--fused-q", action="store_true", help="ARACHNE_FLAG_FWD_FUSED_Q: RMSNorm + RoPE of the query tiles inside fwd_kernel instead of the prologue (A/B)")
    ap.add_argument("--image-copies", action="store_true", help="ARACHNE_FLAG_IMAGE_COPIES: the prologue copies V / dO into tile images (round-1 path) instead of tensor-map TMA from the raw tensors (A/B)")
    ap.add_argument("--heads", type=int, default=0, help="override the head count: the per-rank share of a Ulysses group of degree H/heads")
    ap.add_argument("--seed-offset", type=int, default=0, help="heavytail: another batch drawn from the same recipe (R18)")
    ap.add_argument("--sp", default="none", choices=["none", "ulysses", "cp"],
                    help="N > 1: strong scaling of ONE batch over the N GPUs with sequence parallelism (peer memory, fused All-to-All)")
    ap.add_argument("--src-hash", action="store_true", help="print the kernel source hash (for profiles/r2_traffic.csv) and exit")
    args = ap.parse_args()
    if args.src_hash:
        print(kernel_source_hash())
        return
    if needs_self_launch(args, os.environ):
        # plain `python bench.py --gpus N`: become the launcher of N ranks (each re-enters main() with WORLD_SIZE set)
        raise SystemExit(self_launch(args, sys.argv[1:]))
    if args.impl == "reference":
        return run_reference(args)
    if args.sp != "none":
        from paper_2607_01701_b200 import sp_bench
        return sp_bench.run(args)

    env = Env()
    torch = env.torch
    if env.world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but {env.world} rank(s) are running (WORLD_SIZE): the line's n_gpus must be "
                         f"the number of GPUs that did the work")
    from paper_2607_01701_b200 import binding

    # Multi-GPU (§8 e): sequences/batches are independent -> each rank owns one batch of the same
    # structure (weak scaling), no data-path collective; NCCL only for the barrier and the max-time.
    r = time_workload(env, args.workload, args.steps, args.warmup, deterministic=args.deterministic, order=args.order,
                      seed_offset=args.seed_offset, heads=args.heads, keep=True,
                      extra_flags=(binding.FLAG_FWD_CTA_PAIRS if args.fwd_pairs else 0) | (binding.FLAG_IMAGE_COPIES if args.image_copies else 0) | (binding.FLAG_FWD_MULTICAST if args.fwd_mcast else 0) | (binding.FLAG_FWD_FUSED_Q if args.fused_q else 0))
    r["world"] = env.world
    st, plan, t, flops = r["st"], r["plan"], r["t"], r["flops"]
    s2 = flops / (14.0 * st["D"] * st["H"])

    # ---- e2e through the C-ABI host entry point (pinned host buffers; H2D/D2H inside the timed region)
    e2e = None
    del r["ws"]                      # the main leg's workspace: the e2e call and the target legs bring their own
    torch.cuda.empty_cache()
    if not args.no_e2e:
        nb = t["q"].numel() * 2
        hq, hk, hv, hdo = (x.cpu().pin_memory() for x in (t["q"], t["k"], t["v"], t["dO"]))
        ho, hdq, hdk, hdv = (torch.empty_like(hq).pin_memory() for _ in range(4))
        hlse = torch.empty((plan.H, plan.N), dtype=torch.float32).pin_memory()
        binding.arachne_varlen_attn_fwd_bwd_host(plan, hq, hk, hv, hdo, ho, hlse, hdq, hdk, hdv)   # warm-up (allocates the plan's device buffers)
        env.barrier()
        n_e2e = max(5, min(args.steps, 20))
        dts = []
        for _ in range(n_e2e):
            t0 = time.perf_counter()
            binding.arachne_varlen_attn_fwd_bwd_host(plan, hq, hk, hv, hdo, ho, hlse, hdq, hdk, hdv)   # returns after its own sync
            dts.append(time.perf_counter() - t0)
        dts.sort()
        dt = env.max_over_ranks(dts[len(dts) // 2])
        e2e = {"value": env.world * flops / dt / 1e12, "unit": UNIT, "h2d_bytes_per_step": 4 * nb,
               "d2h_bytes_per_step": 4 * nb + hlse.numel() * 4, "ms_per_step": dt * 1e3, "reps": n_e2e, "stat": "median",
               "ms_min": dts[0] * 1e3, "ms_max": dts[-1] * 1e3,
               "api": "arachne_varlen_attn_fwd_bwd_host (pinned host buffers)"}
        del hq, hk, hv, hdo, ho, hdq, hdk, hdv

    peaks = load_peaks()
    # ---- both north_star targets (and the deterministic backward) in the same record
    targets = None
    if not args.no_targets and args.workload == "long720p" and not args.deterministic and not args.heads:
        tc_main = {k: x.cpu() for k, x in t.items()} if (env.rank == 0 and not args.no_cpu_baseline) else None
        for k in list(t):
            del t[k]
        plan_main_closed = True
        plan.close()
        torch.cuda.empty_cache()
        targets = {"long720p": target_entry(r, peaks, 60.0)}
        ht = time_workload(env, "heavytail", 5, 3); ht["world"] = env.world
        targets["heavytail"] = target_entry(ht, peaks, 50.0)
        targets["heavytail"]["roofline"] = roofline_block(ht, peaks) if env.rank == 0 else None
        torch.cuda.empty_cache()
        det = time_workload(env, "long720p", 3, 3, deterministic=True); det["world"] = env.world
        targets["long720p_deterministic"] = target_entry(det, peaks, 60.0)
        torch.cuda.empty_cache()
    else:
        tc_main = {k: x.cpu() for k, x in t.items()} if (env.rank == 0 and not args.no_cpu_baseline) else None
        plan_main_closed = False

    if env.rank != 0:
        if env.world > 1:
            env.dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel: dense contraction -> tensor roofline.
    roofline = roofline_block(r, peaks)

    cpu = None
    if not args.no_cpu_baseline:
        from oracle import arachne_oracle as orc
        orc.build()
        L_max = max(st["cu_seqlens"][i + 1] - st["cu_seqlens"][i] for i in range(len(st["grids"])))
        # ~10-20 s of oracle time: rows x 2 heads x L_max ~ 2e7 query-row x key products
        v_, dt_, desc, cores = oracle_sample(st, tc_main, budget_rows=max(8, min(L_max, int(8.0e7 / L_max))), heads=2)
        cpu = {"value": v_, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    out = {
        "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": env.world, "steps": args.steps, "warmup": r["warmup"],
        "ms_per_step": r["ms_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic",
        "config": {"workload": args.workload, "order": args.order, "seed_offset": args.seed_offset, "plan_create_ms": round(r["plan_ms"], 3),
                   "deterministic_bwd": bool(args.deterministic), "num_seqs": len(st["grids"]), "total_tokens": st["N"],
                   "heads": st["H"], "head_dim": st["D"], "flop_per_step": flops,
                   "operands": "Q^,K^ fp16 (fwd and bwd recompute), dS fp16 x 2^k, P,V,dO bf16, fp32 accumulate",
                   "l2": "inputs larger than L2 (4 x %.0f MB bf16 tensors + tiled workspace)" % r["tensor_mb"],
                   "pct_of_measured_bf16_burst": 100.0 * r["value"] / env.world / peaks["burst"],
                   "pct_of_measured_bf16_sustained": 100.0 * r["value"] / env.world / peaks["sustained"],
                   "pct_of_nominal_2250": 100.0 * r["value"] / env.world / 2250.0,
                   "fwd_ms": sum(ms for _, ms in r["kt_f"]), "bwd_ms": sum(ms for _, ms in r["kt_b"]),
                   "targets": targets},
        "cta_balance": r["cta_balance"], "clocks": r["clocks"], "e2e": e2e, "gpu_launches": r["launches"], "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    if not plan_main_closed:
        plan.close()
    if env.world > 1:
        env.dist.destroy_process_group()


if __name__ == "__main__":
    main()
