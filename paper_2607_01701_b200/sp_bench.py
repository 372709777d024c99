"""bench.py --sp ulysses|cp : STRONG scaling of one packed batch over the N GPUs of a node with sequence parallelism.

The data-parallel replica mode of bench.py (weak scaling, no data-path collective) is the metric's multi-GPU form (DESIGN.md
§9).  This mode exercises the other way the path shards: ONE batch, token-range shards in
peer-visible memory, the All-to-All (Ulysses) or the K/V exchange and dK/dV reduce-scatter (context parallelism) folded into the
kernels as peer loads / stores over NVLink — `ulysses.UlyssesAttention` / `context_parallel.ContextParallelAttention`.

Launch exactly like bench.py (torchrun, one rank per GPU, NCCL).  Rank barriers: host sync + group barrier by default,
stream-ordered with ARACHNE_SP_BARRIER=stream (ulysses.RankSync; opt-in until it has run on >= 2 GPUs); shards live
in symmetric memory.  When the node exposes fewer GPUs than ranks (this pool: one), the ranks share device 0, barriers fall
back to gloo and shards to CUDA IPC — a functional check of the same code path, not a scaling number (`config.emulated`).
Holds no attention arithmetic.
"""
from __future__ import annotations

import json
import os
import time


def run(args):
    import torch
    import torch.distributed as dist

    from . import context_parallel, inputs, ulysses

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    n_dev = torch.cuda.device_count()
    if n_dev == 0:
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback")
    emulated = n_dev < world                       # several ranks on one device: no NCCL, no symmetric memory
    torch.cuda.set_device(local_rank % n_dev)
    dev = torch.device("cuda", local_rank % n_dev)
    if emulated:
        dist.init_process_group("gloo")
    else:
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log shows the rank count and NVLS
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=dev)
    transport = "ipc" if emulated else "symm"

    st = inputs.structure(args.workload, order=args.order, seed_offset=args.seed_offset)
    st["name"] = args.workload
    if args.sp == "ulysses":
        drv = ulysses.UlyssesAttention(st, transport=transport)
        par = f"ulysses{world}"
    else:
        drv = context_parallel.ContextParallelAttention(st, transport=transport)
        par = f"cp{world}"
    lo, hi = drv.starts[rank], drv.starts[rank + 1]
    for tid, name in ((1, "q"), (2, "k"), (3, "v"), (4, "dO")):
        if hi > lo:      # every rank fills ITS token shard (seeded N(0,1) bf16, its own stream of the generator)
            seed = inputs.BASE_SEED + 16 * st["index"] + tid + 1000 * (rank + 1)
            drv.buf[name].local(hi - lo).copy_(inputs.randn_bf16((hi - lo, st["H"], st["D"]), seed, dev))
    torch.cuda.synchronize()
    dist.barrier()

    def step():
        drv.forward()
        drv.backward()

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    dist.barrier()
    wall_ms = 1e3 * (time.perf_counter() - t0)
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64)
    if emulated:
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    else:
        ms = ms.to(dev)
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_step = float(ms.item()) / args.steps
    flops = inputs.attention_flops(st)                    # ONE batch for the whole group: strong scaling
    if rank == 0:
        print(json.dumps({
            "metric": "varlen 3D attention fwd+bwd TFLOPS", "value": flops / (ms_step * 1e-3) / 1e12, "unit": "TFLOP/s",
            "n_gpus": world, "steps": args.steps, "warmup": warmup, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": {"workload": args.workload, "parallelism": par, "transport": transport, "emulated": emulated,
                       "barrier": drv._sync.describe(),
                       "shard_tokens": [drv.starts[r + 1] - drv.starts[r] for r in range(world)],
                       "num_seqs": len(st["grids"]), "total_tokens": st["N"], "heads": st["H"], "head_dim": st["D"],
                       "flop_per_step": flops, "wall_ms_per_step": wall_ms / args.steps,
                       "nvlink_bytes_per_rank_fwd": ulysses.all_to_all_volume_bytes(st["N"], st["H"], st["D"], world, False) if args.sp == "ulysses" else None,
                       "nvlink_bytes_per_rank_bwd": ulysses.all_to_all_volume_bytes(st["N"], st["H"], st["D"], world, True) if args.sp == "ulysses" else None},
            "gpu_launches": args.steps * (drv.plan.num_launches(False) + drv.plan.num_launches(True) + (2 if args.sp == "cp" else 0)),
        }))
    drv.close()
    dist.destroy_process_group()
