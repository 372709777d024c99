"""Pins for the fp64 oracle (CPU only).  The paper prints no number for this path (it never
specifies the attention arithmetic: PAPER.md:107-113 only names it), so the oracle is pinned to
what the mathematics fixes: an independent brute force, library routines it must reduce to,
closed forms, invariants, and finite differences.  Each test says which mistake it would catch.
"""
import math

import numpy as np
import pytest
import torch

from paper_2607_01701_b200 import inputs

torch.set_num_threads(4)


def tiny_problem(seed=0, grids=((1, 8, 8), (2, 10, 10)), H=2, D=64, scale_inputs=1.0):
    st = inputs.pack(grids, H, D, index=0)
    t = inputs.make_inputs(st)
    rng = np.random.default_rng(seed)
    arr = {k: v.double().numpy() * scale_inputs for k, v in t.items()}
    if seed:
        # non-bf16 perturbation so tests do not depend on bf16-exact inputs
        arr = {k: v + 1e-3 * rng.standard_normal(v.shape) for k, v in arr.items()}
    return st, arr


# --------------------------------------------------------------------------------------------
# 1. brute force, written here from the definition with its own RMSNorm / RoPE lines
#    (catches: any dropped term, wrong pairing, wrong axis slice, wrong scale, wrong position map)
def brute_force(q, k, v, cu, grids, rope_dims, theta=10000.0, eps=1e-6):
    N, H, D = q.shape
    O = np.zeros((N, H, D))
    LSE = np.zeros((H, N))

    def prep(x, n_in_seq, grid):
        T, Hg, Wg = grid
        pos = (n_in_seq // (Hg * Wg), (n_in_seq // Wg) % Hg, n_in_seq % Wg)
        rms = math.sqrt(sum(xx * xx for xx in x) / D + eps)
        y = [xx / rms for xx in x]
        out = list(y)
        base = 0
        for a in range(3):
            da = rope_dims[a]
            for p in range(da // 2):
                ang = pos[a] / (theta ** (2.0 * p / da))
                c, s = math.cos(ang), math.sin(ang)
                a0, a1 = y[base + 2 * p], y[base + 2 * p + 1]
                out[base + 2 * p] = a0 * c - a1 * s
                out[base + 2 * p + 1] = a0 * s + a1 * c
            base += da
        return out

    for b in range(len(cu) - 1):
        s0, e0 = cu[b], cu[b + 1]
        for h in range(H):
            qt = [prep(list(q[n, h]), n - s0, grids[b]) for n in range(s0, e0)]
            kt = [prep(list(k[n, h]), n - s0, grids[b]) for n in range(s0, e0)]
            for i in range(e0 - s0):
                w = [math.exp(sum(a * c for a, c in zip(qt[i], kt[j])) / math.sqrt(D)) for j in range(e0 - s0)]
                Z = sum(w)
                LSE[h, s0 + i] = math.log(Z)
                for j in range(e0 - s0):
                    O[s0 + i, h] += (w[j] / Z) * v[s0 + j, h]
    return O, LSE


def test_brute_force_tiny(orc):
    st, a = tiny_problem(seed=3, grids=((1, 3, 4), (2, 3, 5)), H=2, D=64)
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"])
    O, LSE = brute_force(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], st["rope_dims"])
    assert np.max(np.abs(ref["O"] - O)) <= 1e-12
    assert np.max(np.abs(ref["LSE"] - LSE)) <= 1e-12


def test_brute_force_other_split_D128(orc):
    st = inputs.pack([(2, 2, 3)], 1, 128, rope_dims=(16, 56, 56))
    a = {k: v.double().numpy() for k, v in inputs.make_inputs(st).items()}
    ref = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], rope_dims=(16, 56, 56))
    O, LSE = brute_force(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], (16, 56, 56))
    assert np.max(np.abs(ref["O"] - O)) <= 1e-12 and np.max(np.abs(ref["LSE"] - LSE)) <= 1e-12


# --------------------------------------------------------------------------------------------
# 2. softmax: rows of P sum to 1; V == const => O == const  (catches a wrong normaliser)
def test_softmax_rows_sum_to_one_and_constant_V(orc):
    st, a = tiny_problem()
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], want_P=True)
    for P in r["P"].values():
        assert np.max(np.abs(P.sum(axis=1) - 1.0)) <= 1e-14
        assert P.min() >= 0.0
    v = np.ones_like(a["v"]) * np.arange(1, st["D"] + 1)[None, None, :]
    r = orc.attention(a["q"], a["k"], v, st["cu_seqlens"], st["grids"])
    assert np.max(np.abs(r["O"] - v)) <= 1e-12


# --------------------------------------------------------------------------------------------
# 3. block-diagonality: packed == each sequence alone (bitwise); poisoning the OTHER sequence
#    changes nothing (catches cross-sequence leaks and wrong cu_seqlens offsets)
def test_packed_equals_separate_and_poison(orc):
    st, a = tiny_problem()
    cu = st["cu_seqlens"]
    full = orc.attention(a["q"], a["k"], a["v"], cu, st["grids"], dO=a["dO"])
    for b in range(2):
        s, e = cu[b], cu[b + 1]
        one = orc.attention(a["q"][s:e], a["k"][s:e], a["v"][s:e], [0, e - s], [st["grids"][b]], dO=a["dO"][s:e])
        for key in ("O", "dQ", "dK", "dV"):
            assert np.array_equal(one[key], full[key][s:e])
        assert np.array_equal(one["LSE"], full["LSE"][:, s:e])
    p = {k: v.copy() for k, v in a.items()}
    for k in ("q", "k", "v", "dO"):
        p[k][cu[1]:] = 1.0e4
    poisoned = orc.attention(p["q"], p["k"], p["v"], cu, st["grids"], dO=p["dO"])
    for key in ("O", "dQ", "dK", "dV"):
        assert np.array_equal(poisoned[key][: cu[1]], full[key][: cu[1]])


# 4. order independence: permuting the sequences of the pack permutes the outputs
def test_permutation_of_sequences(orc):
    st, a = tiny_problem()
    cu = st["cu_seqlens"]
    full = orc.attention(a["q"], a["k"], a["v"], cu, st["grids"], dO=a["dO"])
    perm = np.concatenate([np.arange(cu[1], cu[2]), np.arange(cu[0], cu[1])])
    sw = orc.attention(a["q"][perm], a["k"][perm], a["v"][perm], [0, cu[2] - cu[1], cu[2]],
                       st["grids"][::-1], dO=a["dO"][perm])
    for key in ("O", "dQ", "dK", "dV"):
        assert np.array_equal(sw[key], full[key][perm])
    assert np.array_equal(sw["LSE"], full["LSE"][:, perm])


# --------------------------------------------------------------------------------------------
# 5. gradients by central finite differences of l = sum(O * dO) (R12, R13)
#    (catches any error in the backward: sign, missing D_i, missing scale, norm/rope chain rule)
@pytest.mark.parametrize("gamma_mode", ["ones", "random"])
def test_finite_differences(orc, gamma_mode):
    st, a = tiny_problem(seed=5, grids=((1, 3, 4), (2, 2, 3)), H=2, D=64)
    cu, grids = st["cu_seqlens"], st["grids"]
    rng = np.random.default_rng(7)
    gq = gk = None
    if gamma_mode == "random":
        gq, gk = 0.5 + rng.random(64), 0.5 + rng.random(64)
    base = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=a["dO"], gamma_q=gq, gamma_k=gk)

    def loss(q, k, v):
        return float(np.sum(orc.attention(q, k, v, cu, grids, gamma_q=gq, gamma_k=gk)["O"] * a["dO"]))

    hstep = 1e-4
    for name, grad in (("q", base["dQ"]), ("k", base["dK"]), ("v", base["dV"])):
        N = a[name].shape[0]
        coords = [(0, 0, 0), (cu[1] - 1, 1, 63), (cu[1], 0, 17), (N - 1, 1, 40)]
        coords += [tuple(int(x) for x in (rng.integers(N), rng.integers(2), rng.integers(64))) for _ in range(8)]
        for c in coords:
            args = {k: a[k].copy() for k in ("q", "k", "v")}
            args[name][c] += hstep
            lp = loss(**args)
            args[name][c] -= 2 * hstep
            lm = loss(**args)
            fd = (lp - lm) / (2 * hstep)
            assert abs(fd - grad[c]) <= 1e-6 * max(1.0, abs(grad[c])) + 1e-9, (name, c, fd, grad[c])


# --------------------------------------------------------------------------------------------
# 6. reduces to a library routine: norm and RoPE off == torch SDPA in fp64, per sequence
def test_equals_torch_sdpa_when_norm_and_rope_off(orc):
    st, a = tiny_problem(scale_inputs=0.5)
    cu = st["cu_seqlens"]
    r = orc.attention(a["q"], a["k"], a["v"], cu, st["grids"], no_norm=True, no_rope=True)
    for b in range(2):
        s, e = cu[b], cu[b + 1]
        tq, tk, tv = (torch.from_numpy(a[k][s:e]).permute(1, 0, 2)[None] for k in ("q", "k", "v"))
        o = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv)[0].permute(1, 0, 2).numpy()
        assert np.max(np.abs(o - r["O"][s:e])) <= 1e-12
        lse = torch.logsumexp(tq[0] @ tk[0].transpose(1, 2) / math.sqrt(st["D"]), dim=-1).numpy()
        assert np.max(np.abs(lse - r["LSE"][:, s:e])) <= 1e-12


# 6b. third opinion for the whole function incl. gradients: torch fp64 composite + autograd
def torch_composite(q, k, v, cu, grids, rope_dims, gq, gk, theta=10000.0, eps=1e-6):
    N, H, D = q.shape
    outs = []
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        T, Hg, Wg = grids[b]
        n = torch.arange(e - s)
        pos = torch.stack([n // (Hg * Wg), (n // Wg) % Hg, n % Wg], dim=1).double()
        cs, sn = [], []
        for a_, da in enumerate(rope_dims):
            freq = theta ** (-2.0 * torch.arange(da // 2).double() / da)
            ang = pos[:, a_:a_ + 1] * freq[None]
            cs.append(torch.cos(ang)); sn.append(torch.sin(ang))
        cs, sn = torch.cat(cs, 1)[:, None, :], torch.cat(sn, 1)[:, None, :]

        def nr(x, g):
            x = x * torch.rsqrt((x * x).mean(-1, keepdim=True) + eps) * g
            x0, x1 = x[..., 0::2], x[..., 1::2]
            return torch.stack([x0 * cs - x1 * sn, x0 * sn + x1 * cs], dim=-1).flatten(-2)

        qt, kt = nr(q[s:e], gq), nr(k[s:e], gk)
        sc = torch.einsum("ihd,jhd->hij", qt, kt) / math.sqrt(D)
        outs.append(torch.einsum("hij,jhd->ihd", torch.softmax(sc, -1), v[s:e]))
    return torch.cat(outs, 0)


def test_equals_torch_autograd_composite(orc):
    st, a = tiny_problem(seed=11)
    rng = np.random.default_rng(2)
    gq, gk = 0.5 + rng.random(64), 0.5 + rng.random(64)
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], dO=a["dO"], gamma_q=gq, gamma_k=gk)
    tq, tk, tv = (torch.from_numpy(a[k]).requires_grad_(True) for k in ("q", "k", "v"))
    o = torch_composite(tq, tk, tv, st["cu_seqlens"], st["grids"], st["rope_dims"], torch.from_numpy(gq), torch.from_numpy(gk))
    (o * torch.from_numpy(a["dO"])).sum().backward()
    assert np.max(np.abs(o.detach().numpy() - r["O"])) <= 1e-12
    for t, key in ((tq, "dQ"), (tk, "dK"), (tv, "dV")):
        assert np.max(np.abs(t.grad.numpy() - r[key])) <= 1e-10 * max(1.0, np.max(np.abs(r[key])))


# --------------------------------------------------------------------------------------------
# 7. closed forms
def test_closed_form_single_token(orc):
    rng = np.random.default_rng(0)
    q, k, v, dO = (rng.standard_normal((1, 3, 64)) for _ in range(4))
    r = orc.attention(q, k, v, [0, 1], [(1, 1, 1)], dO=dO)
    assert np.allclose(r["O"], v, atol=1e-15)                  # one key => P = 1
    qh = q / np.sqrt((q * q).mean(-1, keepdims=True) + 1e-6)
    kh = k / np.sqrt((k * k).mean(-1, keepdims=True) + 1e-6)
    assert np.allclose(r["LSE"][:, 0], (qh * kh).sum(-1)[0] / 8.0, atol=1e-13)   # RoPE at pos 0 = identity
    assert np.allclose(r["dV"], dO, atol=1e-15)
    assert np.max(np.abs(r["dQ"])) <= 1e-15 and np.max(np.abs(r["dK"])) <= 1e-15


def test_closed_form_zero_query_uniform_attention(orc):
    st, a = tiny_problem()
    cu = st["cu_seqlens"]
    r = orc.attention(np.zeros_like(a["q"]), a["k"], a["v"], cu, st["grids"])
    for b in range(2):
        s, e = cu[b], cu[b + 1]
        assert np.allclose(r["O"][s:e], a["v"][s:e].mean(0, keepdims=True), atol=1e-13)
        assert np.allclose(r["LSE"][:, s:e], math.log(e - s), atol=1e-13)


def test_lse_bound_from_qk_norm(orc):
    st, a = tiny_problem()
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"])
    L = np.repeat(np.diff(st["cu_seqlens"]), np.diff(st["cu_seqlens"]))
    assert np.all(np.abs(r["LSE"] - np.log(L)[None]) <= math.sqrt(st["D"]) + 1e-9)


# --------------------------------------------------------------------------------------------
# 8. RMSNorm is applied per (token, head): scaling a raw row by 2^k leaves O, LSE unchanged and
#    scales that row's gradient by 2^-k (eps = 0 makes it exact); sum_d dQ*Q = 0 (radial direction)
def test_rmsnorm_row_scale_invariance(orc):
    st, a = tiny_problem()
    cu, grids = st["cu_seqlens"], st["grids"]
    r0 = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=a["dO"], eps=0.0)
    q2, k2 = a["q"].copy(), a["k"].copy()
    q2[5, 1] *= 8.0
    k2[70, 0] *= 0.25
    r1 = orc.attention(q2, k2, a["v"], cu, grids, dO=a["dO"], eps=0.0)
    assert np.max(np.abs(r1["O"] - r0["O"])) <= 1e-13 and np.max(np.abs(r1["LSE"] - r0["LSE"])) <= 1e-13
    assert np.allclose(r1["dQ"][5, 1], r0["dQ"][5, 1] / 8.0, rtol=1e-10, atol=1e-15)
    assert np.allclose(r1["dK"][70, 0], r0["dK"][70, 0] * 4.0, rtol=1e-10, atol=1e-15)
    assert np.max(np.abs((r0["dQ"] * a["q"]).sum(-1))) <= 1e-12
    assert np.max(np.abs((r0["dK"] * a["k"]).sum(-1))) <= 1e-12
    # and it is NOT invariant to scaling a single element (norm is over head_dim, not elementwise)
    q3 = a["q"].copy()
    q3[5, 1, 0] *= 8.0
    assert np.max(np.abs(orc.attention(q3, a["k"], a["v"], cu, grids)["O"] - r0["O"])) > 1e-6


# --------------------------------------------------------------------------------------------
# 9. RoPE: preserves the norm; scores depend on position differences only; t/h/w axes use their own
#    slice and position; known rotation of one pair
def test_rope_properties(orc):
    rng = np.random.default_rng(4)
    x = rng.standard_normal(64)
    y = orc.norm_rope(x, (3, 5, 7), no_norm=True)
    assert abs(np.linalg.norm(y) - np.linalg.norm(x)) <= 1e-13
    assert np.array_equal(orc.norm_rope(x, (0, 0, 0), no_norm=True), x)
    # pair p=0 of every axis rotates by exactly pos_a radians (theta^0 = 1)
    for a_, base in enumerate((0, 16, 40)):
        pos = [0, 0, 0]
        pos[a_] = 2
        y = orc.norm_rope(x, pos, no_norm=True)
        c, s = math.cos(2.0), math.sin(2.0)
        assert np.allclose(y[base:base + 2], [x[base] * c - x[base + 1] * s, x[base] * s + x[base + 1] * c], atol=1e-14)
        other = np.ones(64, bool)
        lo, hi = (0, 16) if a_ == 0 else ((16, 40) if a_ == 1 else (40, 64))
        other[lo:hi] = False
        assert np.array_equal(y[other], x[other])              # only that axis' slice moves
    # last pair of the t slice (d_t = 16, p = 7): angle = pos * theta^(-14/16)
    y = orc.norm_rope(x, (5, 0, 0), no_norm=True)
    ang = 5.0 * 10000.0 ** (-14.0 / 16.0)
    assert np.allclose(y[14], x[14] * math.cos(ang) - x[15] * math.sin(ang), atol=1e-14)


def test_rope_shift_invariance_and_axis_distinguishability(orc):
    st, a = tiny_problem(grids=((2, 3, 4),), H=2, D=64)
    cu, grids = st["cu_seqlens"], st["grids"]
    r0 = orc.attention(a["q"], a["k"], a["v"], cu, grids)
    r1 = orc.attention(a["q"], a["k"], a["v"], cu, grids, pos_offset=(7, 11, 13))
    assert np.max(np.abs(r0["O"] - r1["O"])) <= 1e-12 and np.max(np.abs(r0["LSE"] - r1["LSE"])) <= 1e-12
    # transposing the (h, w) grid, re-ordering tokens and swapping the (equal-width) h/w slices
    # of head_dim permutes the outputs
    T, Hg, Wg = grids[0]
    idx = np.arange(T * Hg * Wg).reshape(T, Hg, Wg).transpose(0, 2, 1).reshape(-1)   # new order: (t, w, h)
    dperm = np.concatenate([np.arange(16), np.arange(40, 64), np.arange(16, 40)])
    q2, k2 = a["q"][idx][:, :, dperm], a["k"][idx][:, :, dperm]
    r2 = orc.attention(q2, k2, a["v"][idx], cu, [(T, Wg, Hg)])
    assert np.max(np.abs(r2["O"] - r0["O"][idx])) <= 1e-12
    # without swapping the slices the result differs: h and w are distinguishable
    r3 = orc.attention(a["q"][idx], a["k"][idx], a["v"][idx], cu, [(T, Wg, Hg)])
    assert np.max(np.abs(r3["O"] - r0["O"][idx])) > 1e-4
    # and a flat 1D position reading (all on one axis) also differs
    r4 = orc.attention(a["q"], a["k"], a["v"], cu, [(T * Hg * Wg, 1, 1)])
    assert np.max(np.abs(r4["O"] - r0["O"])) > 1e-4


# --------------------------------------------------------------------------------------------
# 10. sum_j dV_j = sum_i dO_i per (sequence, head)  (follows from rows of P summing to 1)
def test_dV_column_sum(orc):
    st, a = tiny_problem()
    cu = st["cu_seqlens"]
    r = orc.attention(a["q"], a["k"], a["v"], cu, st["grids"], dO=a["dO"])
    for b in range(2):
        s, e = cu[b], cu[b + 1]
        assert np.max(np.abs(r["dV"][s:e].sum(0) - a["dO"][s:e].sum(0))) <= 1e-12


# 11. row-subset mode: O/LSE/dQ of sampled rows == full run; dK/dV == full run on masked dO; linearity
def test_row_subset_and_masked_dO(orc):
    st, a = tiny_problem()
    cu, grids = st["cu_seqlens"], st["grids"]
    rows = inputs.sample_rows(st, per_seq=6, seed=1)
    sub = orc.attention_rows(a["q"], a["k"], a["v"], cu, grids, rows, dO=a["dO"])
    full = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=a["dO"])
    assert np.max(np.abs(sub["O"] - full["O"][rows])) <= 1e-14
    assert np.max(np.abs(sub["LSE"] - full["LSE"][:, rows])) <= 1e-14
    assert np.max(np.abs(sub["dQ"] - full["dQ"][rows])) <= 1e-14
    dOm = np.zeros_like(a["dO"])
    dOm[rows] = a["dO"][rows]
    masked = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=dOm)
    assert np.max(np.abs(sub["dK"] - masked["dK"])) <= 1e-14
    assert np.max(np.abs(sub["dV"] - masked["dV"])) <= 1e-14
    rest = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=a["dO"] - dOm)
    for key in ("dQ", "dK", "dV"):
        assert np.max(np.abs(masked[key] + rest[key] - full[key])) <= 1e-13


def test_rejects_bad_packing(orc):
    st, a = tiny_problem()
    with pytest.raises(AssertionError):
        orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], [(1, 8, 8), (2, 10, 11)])
    with pytest.raises(AssertionError):
        orc.attention(a["q"], a["k"], a["v"], [0, 64, 64, 264], [(1, 8, 8), (1, 1, 1), (2, 10, 10)])
