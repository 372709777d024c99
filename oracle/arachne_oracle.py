"""fp64 CPU oracle for packed varlen 3D attention — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2607_01701_b200 and the product path
never imports it.

The arithmetic lives in arachne_oracle.c (one (sequence, head) problem on fp64 arrays, the
plain definition; see its header for the passages and readings it follows).  This wrapper
only does the bookkeeping of the packed layout (BASELINE.json north_star: "packed batch ...
block-diagonal so no token attends across sequences"): it slices sequence b / head h out of
the [N, H, D] tensors, calls the C routine, and scatters the results back.  Sequences and
heads are independent, so the loop over them IS the block-diagonal definition (R11).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "arachne_oracle.c")
_LIB = os.path.join(_HERE, "libarachne_oracle.so")


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, OpenMP).  No -ffast-math: fp64 semantics as written."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Cfg(ctypes.Structure):
    _fields_ = [
        ("D", ctypes.c_int),
        ("rope_dims", ctypes.c_int * 3),
        ("theta", ctypes.c_double),
        ("eps", ctypes.c_double),
        ("scale", ctypes.c_double),
        ("no_norm", ctypes.c_int),
        ("no_rope", ctypes.c_int),
        ("pos_offset", ctypes.c_int * 3),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.arachne_oracle_head.restype = ctypes.c_int
        lib.arachne_oracle_head.argtypes = [ctypes.POINTER(_Cfg), ip, ctypes.c_int, ctypes.c_int, ip] + [dp] * 12
        lib.arachne_oracle_head_joint.restype = ctypes.c_int
        lib.arachne_oracle_head_joint.argtypes = [ctypes.POINTER(_Cfg), ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ip] + [dp] * 14
        lib.arachne_oracle_norm_rope.restype = ctypes.c_int
        lib.arachne_oracle_norm_rope.argtypes = [ctypes.POINTER(_Cfg), ip, dp, dp, dp]
        lib.arachne_oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().arachne_oracle_num_threads())


def default_rope_dims(D: int):
    """R6: (16,24,24) for D=64 (BASELINE.json configs[0]); doubled, (32,48,48), for D=128."""
    return {64: (16, 24, 24), 128: (32, 48, 48)}[D]


def _cfg(D, rope_dims=None, theta=10000.0, eps=1e-6, scale=None, no_norm=False, no_rope=False,
         pos_offset=(0, 0, 0)) -> _Cfg:
    rope_dims = tuple(rope_dims) if rope_dims is not None else default_rope_dims(D)
    assert sum(rope_dims) == D and all(r % 2 == 0 for r in rope_dims)
    c = _Cfg()
    c.D = D
    c.rope_dims[:] = rope_dims
    c.theta = float(theta)
    c.eps = float(eps)
    c.scale = float(scale) if scale else 1.0 / np.sqrt(D)   # R8
    c.no_norm = int(no_norm)
    c.no_rope = int(no_rope)
    c.pos_offset[:] = pos_offset
    return c


def _dptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _iptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def norm_rope(x, pos, gamma=None, **kw):
    """x~ of a single row (debug hook for the RMSNorm / RoPE pins)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    D = x.shape[0]
    g = np.ones(D) if gamma is None else np.ascontiguousarray(gamma, dtype=np.float64)
    out = np.empty(D)
    p = np.asarray(pos, dtype=np.int32)
    _load().arachne_oracle_norm_rope(ctypes.byref(_cfg(D, **kw)), _iptr(p), _dptr(x), _dptr(g), _dptr(out))
    return out


def head(q_rows, k, v, grid, qidx=None, dO_rows=None, gamma_q=None, gamma_k=None, want_P=False, n_text=0, **kw):
    """One (sequence, head) problem.  q_rows [R,D], k,v [L,D], grid=(T,Hg,Wg), qidx [R] in-sequence
    token indices of the query rows (default: all L rows).  n_text: the last n_text of the L tokens are
    text tokens (R21: normed, not rotated).  Returns a dict of fp64 arrays; with dO_rows also dGq, dGk [D]
    (R22: this problem's terms of dl/dgamma_q, dl/dgamma_k)."""
    k = np.ascontiguousarray(k, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    q_rows = np.ascontiguousarray(q_rows, dtype=np.float64)
    L, D = k.shape
    R = q_rows.shape[0]
    qidx = np.arange(L, dtype=np.int32) if qidx is None else np.ascontiguousarray(qidx, dtype=np.int32)
    assert qidx.shape[0] == R
    gq = np.ones(D) if gamma_q is None else np.ascontiguousarray(gamma_q, dtype=np.float64)
    gk = np.ones(D) if gamma_k is None else np.ascontiguousarray(gamma_k, dtype=np.float64)
    g = np.asarray(grid, dtype=np.int32)
    out = {"O": np.empty((R, D)), "LSE": np.empty(R)}
    P = np.empty((R, L)) if want_P else None
    dO = dQ = dK = dV = None
    if dO_rows is not None:
        dO = np.ascontiguousarray(dO_rows, dtype=np.float64)
        dQ, dK, dV = np.empty((R, D)), np.empty((L, D)), np.empty((L, D))
        dGq, dGk = np.empty(D), np.empty(D)
    else:
        dGq = dGk = None
    rc = _load().arachne_oracle_head_joint(
        ctypes.byref(_cfg(D, **kw)), _iptr(g), int(n_text), L, R, _iptr(qidx), _dptr(q_rows), _dptr(k), _dptr(v),
        _dptr(gq), _dptr(gk), _dptr(dO), _dptr(out["O"]), _dptr(out["LSE"]), _dptr(P), _dptr(dQ),
        _dptr(dK), _dptr(dV), _dptr(dGq), _dptr(dGk))
    if rc != 0:
        raise ValueError("arachne_oracle_head rejected its arguments (L>=1, grid product + n_text == L)")
    if want_P:
        out["P"] = P
    if dO is not None:
        out.update(dQ=dQ, dK=dK, dV=dV, dGq=dGq, dGk=dGk)
    return out


def _check_packing(cu_seqlens, grids, N, text_lens=None):
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    grids = np.asarray(grids, dtype=np.int64).reshape(-1, 3)
    text = np.zeros(len(cu) - 1, dtype=np.int64) if text_lens is None else np.asarray(text_lens, dtype=np.int64)
    assert cu[0] == 0 and np.all(np.diff(cu) >= 1) and cu[-1] == N, "bad cu_seqlens (R16: L_b >= 1)"
    assert np.all(text >= 0) and np.all(grids.prod(axis=1) + text == np.diff(cu)), "grid product + text != sequence length"
    return cu, grids, text


def attention(q, k, v, cu_seqlens, grids, dO=None, gamma_q=None, gamma_k=None, want_P=False, text_lens=None, **kw):
    """Full packed problem.  q,k,v (and dO) are [N,H,D] arrays of exact input values (any float
    dtype; converted to fp64).  text_lens [B]: trailing text tokens of each sequence (R21; default none).
    Returns O [N,H,D], LSE [H,N] and, if dO is given, dQ,dK,dV [N,H,D] and dGq,dGk [D] (R22: summed over
    sequences and heads in index order)."""
    q, k, v = (np.asarray(a, dtype=np.float64) for a in (q, k, v))
    N, H, D = q.shape
    cu, grids, text = _check_packing(cu_seqlens, grids, N, text_lens)
    res = {"O": np.empty((N, H, D)), "LSE": np.empty((H, N))}
    if dO is not None:
        dO = np.asarray(dO, dtype=np.float64)
        res.update(dQ=np.empty((N, H, D)), dK=np.empty((N, H, D)), dV=np.empty((N, H, D)), dGq=np.zeros(D), dGk=np.zeros(D))
    if want_P:
        res["P"] = {}
    for b in range(len(cu) - 1):
        s, e = int(cu[b]), int(cu[b + 1])
        for h in range(H):
            r = head(q[s:e, h], k[s:e, h], v[s:e, h], grids[b], dO_rows=None if dO is None else dO[s:e, h],
                     gamma_q=gamma_q, gamma_k=gamma_k, want_P=want_P, n_text=int(text[b]), **kw)
            res["O"][s:e, h] = r["O"]
            res["LSE"][h, s:e] = r["LSE"]
            if dO is not None:
                res["dQ"][s:e, h], res["dK"][s:e, h], res["dV"][s:e, h] = r["dQ"], r["dK"], r["dV"]
                res["dGq"] += r["dGq"]
                res["dGk"] += r["dGk"]
            if want_P:
                res["P"][(b, h)] = r["P"]
    return res


def attention_rows(q, k, v, cu_seqlens, grids, rows, dO=None, heads=None, gamma_q=None, gamma_k=None,
                   text_lens=None, **kw):
    """Sampled-row evaluation for configs too large for the O(L^2) run.

    rows : sorted global token indices (any subset).  heads : list of heads (default all).
    Returns O_rows [R,Hs,D], LSE_rows [Hs,R] exactly (a query row needs only its own row of S) and,
    if dO is given, dQ_rows [R,Hs,D] exactly plus dK, dV [N,Hs,D] and dGq, dGk [D] of the MASKED-dO
    problem (dO zero outside `rows` and outside `heads`), which the GPU can reproduce by running its
    backward on that masked dO.
    dO may be the full [N,H,D] tensor (only `rows` are read) or [R,H,D]."""
    N, H, D = q.shape
    cu, grids, text = _check_packing(cu_seqlens, grids, N, text_lens)
    rows = np.asarray(rows, dtype=np.int64)
    assert np.all(np.diff(rows) > 0)
    heads = list(range(H)) if heads is None else list(heads)
    R, Hs = len(rows), len(heads)
    res = {"O": np.empty((R, Hs, D)), "LSE": np.empty((Hs, R)), "rows": rows, "heads": heads}
    if dO is not None:
        res.update(dQ=np.empty((R, Hs, D)), dK=np.zeros((N, Hs, D)), dV=np.zeros((N, Hs, D)), dGq=np.zeros(D), dGk=np.zeros(D))
        dO_is_full = dO.shape[0] == N and N != R
    for b in range(len(cu) - 1):
        s, e = int(cu[b]), int(cu[b + 1])
        sel = np.nonzero((rows >= s) & (rows < e))[0]
        if len(sel) == 0:
            continue
        qidx = (rows[sel] - s).astype(np.int32)
        for hi, h in enumerate(heads):
            dO_rows = None
            if dO is not None:
                dO_rows = np.asarray(dO[rows[sel], h] if dO_is_full else dO[sel, h], dtype=np.float64)
            r = head(np.asarray(q[rows[sel], h], dtype=np.float64), np.asarray(k[s:e, h], dtype=np.float64),
                     np.asarray(v[s:e, h], dtype=np.float64), grids[b], qidx=qidx, dO_rows=dO_rows,
                     gamma_q=gamma_q, gamma_k=gamma_k, n_text=int(text[b]), **kw)
            res["O"][sel, hi] = r["O"]
            res["LSE"][hi, sel] = r["LSE"]
            if dO is not None:
                res["dQ"][sel, hi] = r["dQ"]
                res["dK"][s:e, hi] = r["dK"]
                res["dV"][s:e, hi] = r["dV"]
                res["dGq"] += r["dGq"]      # masked-dO problem restricted to `heads`
                res["dGk"] += r["dGk"]
    return res
