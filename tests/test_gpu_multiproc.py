"""GPU: the multi-rank DRIVERS (ulysses.UlyssesAttention, context_parallel.ContextParallelAttention) run as real separate
processes with real peer mappings — 2 ranks sharing the one GPU of this pool, shards exchanged through CUDA IPC
(arachne_ipc_*), `gloo` for the barriers (NCCL refuses two ranks on one device; symmetric memory likewise).  Each rank
fills its own token shard, runs forward + backward through the driver and checks ITS shard against the fp64 oracle.
No kernel waits on another rank's kernel: ranks are ordered by host barriers only."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01701_b200 import inputs

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, mode, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import sys
        sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
        import parity_util as pu
        from oracle import arachne_oracle as orc
        from paper_2607_01701_b200 import context_parallel, ulysses
        orc.build()
        st = inputs.pack([(2, 9, 11), (1, 8, 8), (3, 10, 13)], 4, 128, index=6, text_lens=[5, 0, 0])      # 203 + 64 + 390 tokens
        full = inputs.make_inputs(st, device="cuda")
        rng = np.random.default_rng(8)
        gq, gk = ((0.5 + rng.random(128)).astype(np.float32) for _ in range(2))
        tgq, tgk = torch.as_tensor(gq, device="cuda"), torch.as_tensor(gk, device="cuda")
        drv = (ulysses.UlyssesAttention(st, transport="ipc") if mode == "ulysses"
               else context_parallel.ContextParallelAttention(st, transport="ipc"))
        lo, hi = drv.starts[rank], drv.starts[rank + 1]
        for name in ("q", "k", "v", "dO"):
            drv.buf[name].local(hi - lo).copy_(full[name][lo:hi])
        for name in ("o", "dq", "dk", "dv"):
            drv.buf[name].local_full.fill_(7.0)
        torch.cuda.synchronize()
        o = drv.forward(tgq, tgk)
        dq, dk, dv, dgq, dgk = drv.backward(tgq, tgk, with_dgamma=True)      # both drivers return the all-reduced dgamma
        torch.cuda.synchronize()
        a = {n: v.float().cpu().numpy().astype(np.float64) for n, v in full.items()}
        ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], gamma_q=gq, gamma_k=gk,
                            rope_dims=st["rope_dims"], text_lens=st["text_lens"])
        for got, key, tol in ((o, "O", 1e-2), (dq, "dQ", 2e-2), (dk, "dK", 2e-2), (dv, "dV", 2e-2)):
            r = pu.rel_l2(pu.to_np(got), ref[key][lo:hi])
            assert r <= tol, (mode, rank, key, r)
        assert pu.rel_l2(pu.to_np(dgq), ref["dGq"]) <= 2e-2 and pu.rel_l2(pu.to_np(dgk), ref["dGk"]) <= 2e-2, (mode, rank)
        drv.close()
        open(os.path.join(out_dir, f"ok_{mode}_{rank}"), "w").write("ok")
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
@pytest.mark.parametrize("mode", ["ulysses", "cp"])
def test_two_processes_one_gpu_ipc_shards(tmp_path, mode):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, mode, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / f"ok_{mode}_0").read_text() == "ok" and (tmp_path / f"ok_{mode}_1").read_text() == "ok"


@pytest.mark.timeout(600)
@pytest.mark.parametrize("sp", ["ulysses", "cp"])
def test_bench_sp_mode_two_ranks_on_one_gpu(sp):
    """`bench.py --gpus 2 --sp ulysses|cp` launched the way the driver launches multi-GPU runs (torch.distributed.run).  With one
    GPU on the box the two ranks share it (gloo barriers, CUDA IPC shards: config.emulated) — a functional check of the
    strong-scaling mode, not a scaling number."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(root, "bench.py"), "--gpus", "2", "--sp", sp, "--workload", "bucket256",
           "--steps", "2", "--warmup", "3"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=500, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [x for x in out.stdout.splitlines() if x.startswith("{")][-1]
    d = json.loads(line)
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["value"] > 0
    assert d["config"]["parallelism"] == f"{sp}2" and d["config"]["emulated"] == (torch.cuda.device_count() < 2)
    print(sp, round(d["value"], 1), "TFLOP/s", d["config"])
