"""Thin ctypes binding over libarachne_sched.so (include/arachne_sched.h): list scheduler + genetic algorithm of the
paper's cascade planner, fed by costmodel.py's Eq. 9 coefficients measured on this repository's
attention kernels.  Argument marshalling only; raises if the library has not been built."""
from __future__ import annotations

import ctypes
import os

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "libarachne_sched.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_2607_01701_b200.build`")
_lib = ctypes.CDLL(_LIB_PATH)

EXPORTS = ["arachne_list_schedule", "arachne_ga_schedule", "arachne_sched_uniform"]
_dp, _ip, _bp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_uint8)
_lib.arachne_list_schedule.restype = ctypes.c_int
_lib.arachne_list_schedule.argtypes = [ctypes.c_int32, _dp, _ip, _ip, _ip, ctypes.c_int32, _dp, _dp, _dp]
_lib.arachne_ga_schedule.restype = ctypes.c_int
_lib.arachne_ga_schedule.argtypes = [ctypes.c_int32, ctypes.c_int32, _ip, _dp, _bp, _ip, _ip, ctypes.c_int32, ctypes.c_int32,
                                     ctypes.c_int32, ctypes.c_double, ctypes.c_int32, ctypes.c_uint64, _ip, _dp, _dp, _dp, _dp]
_lib.arachne_sched_uniform.restype = ctypes.c_double
_lib.arachne_sched_uniform.argtypes = [ctypes.c_uint64] * 5

_ERR = {1: "null pointer", 2: "bad argument", 3: "a cascade has no feasible degree", 4: "dependency cycle / bad predecessor"}


class SchedError(RuntimeError):
    def __init__(self, status):
        self.status = status
        super().__init__(f"arachne_sched status {status}: {_ERR.get(status, 'unknown')}")


def _csr(preds):
    ptr, idx = [0], []
    for p in preds:
        idx.extend(int(x) for x in p)
        ptr.append(len(idx))
    return (ctypes.c_int32 * len(ptr))(*ptr), (ctypes.c_int32 * max(len(idx), 1))(*idx)


def uniform(seed, gen, child, gene, purpose) -> float:
    return float(_lib.arachne_sched_uniform(seed, gen, child, gene, purpose))


def list_schedule(lat, deg, preds, N):
    """-> (start[], end[], makespan)"""
    n = len(lat)
    ptr, idx = _csr(preds)
    s, e, T = (ctypes.c_double * n)(), (ctypes.c_double * n)(), ctypes.c_double()
    rc = _lib.arachne_list_schedule(n, (ctypes.c_double * n)(*lat), (ctypes.c_int32 * n)(*deg), ptr, idx, N, s, e, ctypes.byref(T))
    if rc:
        raise SchedError(rc)
    return list(s), list(e), T.value


def genetic(K, L, feasible, preds, N, p, G, mu, eps, seed):
    """-> (T*, best chromosome (index into K per cascade), start[], end[], history[G])"""
    n, nk = len(L), len(K)
    ptr, idx = _csr(preds)
    flatL = (ctypes.c_double * (n * nk))(*[float(x) for row in L for x in row])
    flatF = (ctypes.c_uint8 * (n * nk))(*[1 if x else 0 for row in feasible for x in row])
    best, s, e = (ctypes.c_int32 * n)(), (ctypes.c_double * n)(), (ctypes.c_double * n)()
    T, hist = ctypes.c_double(), (ctypes.c_double * G)()
    rc = _lib.arachne_ga_schedule(n, nk, (ctypes.c_int32 * nk)(*K), flatL, flatF, ptr, idx, N, p, G, mu, eps, seed, best, s, e,
                                  ctypes.byref(T), hist)
    if rc:
        raise SchedError(rc)
    return T.value, list(best), list(s), list(e), list(hist)


def dit_instance(st, alpha1_ms, alpha2_ms, n_layers=60, degrees=(1, 2, 4, 8), num_gpus=16, passes=3.0,
                 nvlink_gbs=900.0, max_tokens_per_gpu=70000):
    """One DiT cascade per sequence of the packing structure `st`, latencies from Eq. 9 with the
    coefficients costmodel.fit_alpha measured on this repository's attention (per layer, fwd+bwd; `passes` = 3 counts the
    recompute forward of activation checkpointing, as one more forward ~ 1/3.5 of fwd+bwd is ignored:
    a planning input, not a measurement), V_comm = the Ulysses All-to-All volume of ulysses.all_to_all_volume_bytes over
    BW_eff = NVLink.  Memory (Eq. 8's activation term): tokens / k <= max_tokens_per_gpu.  Seconds."""
    from . import costmodel, ulysses

    cu = st["cu_seqlens"]
    K = [int(k) for k in degrees]
    L, feas = [], []
    for b in range(len(cu) - 1):
        S = cu[b + 1] - cu[b]
        row, ok = [], []
        for k in K:
            comm = 0.0
            if k > 1 and st["H"] % k == 0:
                comm = (ulysses.all_to_all_volume_bytes(S, st["H"], st["D"], k, False) * 2 +
                        ulysses.all_to_all_volume_bytes(S, st["H"], st["D"], k, True)) / (nvlink_gbs * 1e9) * 1e3
            row.append(n_layers * costmodel.predict(alpha1_ms, alpha2_ms, 1, S, k=k, v_comm=comm, bw_eff=1.0) / 1e3)
            ok.append(S / k <= max_tokens_per_gpu and st["H"] % k == 0)
        if not any(ok):
            ok[-1] = True
        L.append(row); feas.append(ok)
    return dict(K=K, L=L, feasible=feas, preds=[[] for _ in L], N=num_gpus)


def main():
    """Plan the heavy-tailed batch (BASELINE.json configs[4]) on 16 GPUs with the measured Eq. 9 coefficients."""
    from . import inputs

    a1, a2 = 5.30e-5, 3.81e-8                       # profiles/r1_alpha_fit.md (ms per token, ms per token^2; one layer, fwd+bwd)
    st = inputs.structure("heavytail")
    inst = dit_instance(st, a1, a2)
    n = len(inst["L"])
    print(f"{n} DiT cascades, {inst['N']} GPUs, degrees {inst['K']}")
    for name, pick in (("static k = 4 (DP4 x SP4)", 2), ("static k = 8", 3)):
        ch = [pick if inst["feasible"][c][pick] else max(j for j in range(len(inst["K"])) if inst["feasible"][c][j]) for c in range(n)]
        T = list_schedule([inst["L"][c][ch[c]] for c in range(n)], [inst["K"][ch[c]] for c in range(n)], inst["preds"], inst["N"])[2]
        print(f"  {name}: makespan {T:.2f} s")
    T, ch, s, e, hist = genetic(inst["K"], inst["L"], inst["feasible"], inst["preds"], inst["N"], p=64, G=40, mu=0.05, eps=2, seed=1)
    work = sum(inst["L"][c][ch[c]] * inst["K"][ch[c]] for c in range(n)) / inst["N"]
    print(f"  Alg. 1 (p=64, G=40): makespan {T:.2f} s (first generation {hist[0]:.2f} s; GPU-time / N bound {work:.2f} s)")
    print("  degrees chosen:", {k: sum(1 for c in range(n) if inst['K'][ch[c]] == k) for k in inst["K"]})


if __name__ == "__main__":
    main()
