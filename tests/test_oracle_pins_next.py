"""Pins for the oracle's SURVEY §8(f) extensions (CPU only): joint text tokens (reading R21) and
dgamma_q / dgamma_k (reading R22).  The paper prints nothing for either (PAPER.md:322 only names the
"hybrid dual/single-stream" model, PAPER.md:201 the < 256-token prompt), so they are pinned to an
independent brute force, a torch fp64 autograd composite, finite differences, closed forms and an
invariant of the loss.  Each test says which mistake it would catch.
"""
import math

import numpy as np
import pytest
import torch

from paper_2607_01701_b200 import inputs

torch.set_num_threads(4)


def joint_problem(seed=1, grids=((1, 3, 4), (2, 2, 3)), text_lens=(5, 3), H=2, D=64):
    st = inputs.pack(grids, H, D, index=0, text_lens=text_lens)
    rng = np.random.default_rng(seed)
    a = {k: v.double().numpy() + 1e-3 * rng.standard_normal(v.shape) for k, v in inputs.make_inputs(st).items()}
    return st, a


# --------------------------------------------------------------------------------------------
# 1. brute force with its own is-text switch (catches: text tokens rotated, text tokens placed before the
#    video tokens, video positions shifted by the text length, text tokens not normed)
def brute_force_joint(q, k, v, cu, grids, text_lens, rope_dims, gq, gk, theta=10000.0, eps=1e-6):
    N, H, D = q.shape
    O, LSE = np.zeros((N, H, D)), np.zeros((H, N))

    def prep(x, g, n, grid):
        T, Hg, Wg = grid
        rms = math.sqrt(sum(xx * xx for xx in x) / D + eps)
        y = [g[d] * x[d] / rms for d in range(D)]
        if n >= T * Hg * Wg:            # text token: no rotation
            return y
        pos = (n // (Hg * Wg), (n // Wg) % Hg, n % Wg)
        out, base = list(y), 0
        for a in range(3):
            da = rope_dims[a]
            for p in range(da // 2):
                ang = pos[a] / (theta ** (2.0 * p / da))
                c, s = math.cos(ang), math.sin(ang)
                out[base + 2 * p] = y[base + 2 * p] * c - y[base + 2 * p + 1] * s
                out[base + 2 * p + 1] = y[base + 2 * p] * s + y[base + 2 * p + 1] * c
            base += da
        return out

    for b in range(len(cu) - 1):
        s0, e0 = cu[b], cu[b + 1]
        for h in range(H):
            qt = [prep(list(q[n, h]), gq, n - s0, grids[b]) for n in range(s0, e0)]
            kt = [prep(list(k[n, h]), gk, n - s0, grids[b]) for n in range(s0, e0)]
            for i in range(e0 - s0):
                w = [math.exp(sum(a * c for a, c in zip(qt[i], kt[j])) / math.sqrt(D)) for j in range(e0 - s0)]
                Z = sum(w)
                LSE[h, s0 + i] = math.log(Z)
                for j in range(e0 - s0):
                    O[s0 + i, h] += (w[j] / Z) * v[s0 + j, h]
    return O, LSE


def test_joint_brute_force(orc):
    st, a = joint_problem()
    rng = np.random.default_rng(3)
    gq, gk = 0.5 + rng.random(64), 0.5 + rng.random(64)
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], text_lens=st["text_lens"], gamma_q=gq, gamma_k=gk)
    O, LSE = brute_force_joint(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], st["text_lens"], st["rope_dims"], gq, gk)
    assert np.max(np.abs(r["O"] - O)) <= 1e-12 and np.max(np.abs(r["LSE"] - LSE)) <= 1e-12


# --------------------------------------------------------------------------------------------
# 2. closed forms.  (a) a video token at the grid origin is not rotated either, so a (1,1,1) grid + n text
#    tokens equals the plain run of n+1 tokens with RoPE off; a text-only sequence (T = 0) likewise.
#    (b) treating the same tokens as video tokens of a (1,1,n+1) grid gives a DIFFERENT result (the switch
#    acts).  (c) text_lens = 0 is the base problem bit for bit.
def test_joint_closed_forms(orc):
    st, a = joint_problem(grids=((1, 1, 1),), text_lens=(7,))
    cu = st["cu_seqlens"]
    r = orc.attention(a["q"], a["k"], a["v"], cu, [(1, 1, 1)], text_lens=[7], dO=a["dO"])
    plain = orc.attention(a["q"], a["k"], a["v"], cu, [(1, 1, 8)], dO=a["dO"], no_rope=True)
    textonly = orc.attention(a["q"], a["k"], a["v"], cu, [(0, 1, 1)], text_lens=[8], dO=a["dO"])
    for key in ("O", "LSE", "dQ", "dK", "dV", "dGq", "dGk"):
        assert np.array_equal(r[key], plain[key]) and np.array_equal(textonly[key], plain[key])
    video = orc.attention(a["q"], a["k"], a["v"], cu, [(1, 1, 8)])
    assert np.max(np.abs(video["O"] - r["O"])) > 1e-4
    st0, a0 = joint_problem(text_lens=(0, 0))
    base = orc.attention(a0["q"], a0["k"], a0["v"], st0["cu_seqlens"], st0["grids"], dO=a0["dO"])
    zero = orc.attention(a0["q"], a0["k"], a0["v"], st0["cu_seqlens"], st0["grids"], dO=a0["dO"], text_lens=[0, 0])
    for key in ("O", "LSE", "dQ", "dK", "dV"):
        assert np.array_equal(base[key], zero[key])


# 3. the video positions do not depend on the text length: appending text tokens whose V is the current
#    output-neutral... simpler and sharper: a text token is position-free, so PERMUTING the text tokens of a
#    sequence permutes the outputs; permuting video tokens does not (catches positions applied to text).
def test_joint_text_tokens_are_position_free(orc):
    st, a = joint_problem(grids=((2, 2, 3),), text_lens=(6,))
    cu, L = st["cu_seqlens"], 18
    r0 = orc.attention(a["q"], a["k"], a["v"], cu, st["grids"], text_lens=[6], dO=a["dO"])
    perm = np.concatenate([np.arange(12), 12 + np.array([3, 0, 5, 1, 4, 2])])
    r1 = orc.attention(a["q"][perm], a["k"][perm], a["v"][perm], cu, st["grids"], text_lens=[6], dO=a["dO"][perm])
    for key in ("O", "dQ", "dK", "dV"):
        assert np.max(np.abs(r1[key] - r0[key][perm])) <= 1e-13
    vperm = np.concatenate([np.array([1, 0]), np.arange(2, L)])
    r2 = orc.attention(a["q"][vperm], a["k"][vperm], a["v"][vperm], cu, st["grids"], text_lens=[6])
    assert np.max(np.abs(r2["O"] - r0["O"][vperm])) > 1e-4


# 4. packed == separate with text (catches text offsets computed from the pack instead of the sequence)
def test_joint_packed_equals_separate(orc):
    st, a = joint_problem()
    cu = st["cu_seqlens"]
    full = orc.attention(a["q"], a["k"], a["v"], cu, st["grids"], text_lens=st["text_lens"], dO=a["dO"])
    dgq, dgk = 0.0, 0.0
    for b in range(2):
        s, e = cu[b], cu[b + 1]
        one = orc.attention(a["q"][s:e], a["k"][s:e], a["v"][s:e], [0, e - s], [st["grids"][b]],
                            text_lens=[st["text_lens"][b]], dO=a["dO"][s:e])
        for key in ("O", "dQ", "dK", "dV"):
            assert np.array_equal(one[key], full[key][s:e])
        dgq, dgk = dgq + one["dGq"], dgk + one["dGk"]
    assert np.allclose(dgq, full["dGq"], rtol=1e-13, atol=1e-15) and np.allclose(dgk, full["dGk"], rtol=1e-13, atol=1e-15)


# --------------------------------------------------------------------------------------------
# 5. third opinion incl. every gradient: torch fp64 composite + autograd (is-text mask written here)
def torch_composite_joint(q, k, v, cu, grids, text_lens, rope_dims, gq, gk, theta=10000.0, eps=1e-6):
    N, H, D = q.shape
    outs = []
    for b in range(len(cu) - 1):
        s, e = cu[b], cu[b + 1]
        T, Hg, Wg = grids[b]
        n = torch.arange(e - s)
        is_video = (n < T * Hg * Wg).double()
        pos = torch.stack([n // (Hg * Wg), (n // Wg) % Hg, n % Wg], dim=1).double() * is_video[:, None]   # text -> origin
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


@pytest.mark.parametrize("text_lens", [(5, 3), (0, 0)])
def test_joint_and_dgamma_equal_torch_autograd(orc, text_lens):
    st, a = joint_problem(seed=11, text_lens=text_lens)
    tl = list(text_lens)
    rng = np.random.default_rng(2)
    gq, gk = 0.5 + rng.random(64), 0.5 + rng.random(64)
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], text_lens=tl, dO=a["dO"], gamma_q=gq, gamma_k=gk)
    tq, tk, tv, tgq, tgk = (torch.from_numpy(x).requires_grad_(True) for x in (a["q"], a["k"], a["v"], gq, gk))
    o = torch_composite_joint(tq, tk, tv, st["cu_seqlens"], st["grids"], tl, st["rope_dims"], tgq, tgk)
    (o * torch.from_numpy(a["dO"])).sum().backward()
    assert np.max(np.abs(o.detach().numpy() - r["O"])) <= 1e-12
    for t, key in ((tq, "dQ"), (tk, "dK"), (tv, "dV"), (tgq, "dGq"), (tgk, "dGk")):
        assert np.max(np.abs(t.grad.numpy() - r[key])) <= 1e-10 * max(1.0, np.max(np.abs(r[key]))), key


# --------------------------------------------------------------------------------------------
# 6. dgamma by central finite differences of l = sum(O * dO) in gamma (catches a missing r, a missing
#    un-rotation, gamma applied twice, a sum over the wrong rows / heads)
def test_dgamma_finite_differences(orc):
    st, a = joint_problem(seed=5)
    cu, grids, tl = st["cu_seqlens"], st["grids"], st["text_lens"]
    rng = np.random.default_rng(7)
    gq, gk = 0.5 + rng.random(64), 0.5 + rng.random(64)
    base = orc.attention(a["q"], a["k"], a["v"], cu, grids, text_lens=tl, dO=a["dO"], gamma_q=gq, gamma_k=gk)

    def loss(gq_, gk_):
        return float(np.sum(orc.attention(a["q"], a["k"], a["v"], cu, grids, text_lens=tl, gamma_q=gq_, gamma_k=gk_)["O"] * a["dO"]))

    h = 1e-4
    for d in (0, 1, 15, 16, 39, 40, 63):
        for which, grad in ((0, base["dGq"]), (1, base["dGk"])):
            gp, gm = [gq.copy(), gk.copy()], [gq.copy(), gk.copy()]
            gp[which][d] += h
            gm[which][d] -= h
            fd = (loss(*gp) - loss(*gm)) / (2 * h)
            assert abs(fd - grad[d]) <= 1e-6 * max(1.0, abs(grad[d])) + 1e-9, (which, d, fd, grad[d])


# 7. invariant: the scores, hence the loss, are unchanged by gamma_q -> c gamma_q, gamma_k -> gamma_k / c,
#    so sum_d gamma_q[d] dGq[d] == sum_d gamma_k[d] dGk[d]; and with RMSNorm off gamma is unused => 0.
def test_dgamma_scaling_invariant_and_no_norm(orc):
    st, a = joint_problem(seed=9)
    rng = np.random.default_rng(1)
    gq, gk = 0.5 + rng.random(64), 0.5 + rng.random(64)
    kw = dict(text_lens=st["text_lens"], dO=a["dO"], gamma_q=gq, gamma_k=gk)
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], **kw)
    lhs, rhs = float(np.dot(gq, r["dGq"])), float(np.dot(gk, r["dGk"]))
    assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(lhs)) and abs(lhs) > 1e-6
    r = orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], no_norm=True, **kw)
    assert np.all(r["dGq"] == 0.0) and np.all(r["dGk"] == 0.0)


# 8. row-subset mode with text + dgamma == full run on the masked dO
def test_joint_row_subset_and_masked_dO(orc):
    st, a = joint_problem()
    cu, grids, tl = st["cu_seqlens"], st["grids"], st["text_lens"]
    rows = inputs.sample_rows(st, per_seq=6, seed=1)
    sub = orc.attention_rows(a["q"], a["k"], a["v"], cu, grids, rows, dO=a["dO"], text_lens=tl)
    dOm = np.zeros_like(a["dO"])
    dOm[rows] = a["dO"][rows]
    masked = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=dOm, text_lens=tl)
    full = orc.attention(a["q"], a["k"], a["v"], cu, grids, dO=a["dO"], text_lens=tl)
    assert np.max(np.abs(sub["O"] - full["O"][rows])) <= 1e-14 and np.max(np.abs(sub["dQ"] - full["dQ"][rows])) <= 1e-14
    for key in ("dK", "dV", "dGq", "dGk"):
        assert np.max(np.abs(sub[key] - masked[key])) <= 1e-13, key


def test_joint_rejects_bad_packing(orc):
    st, a = joint_problem()
    with pytest.raises(AssertionError):
        orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], text_lens=[5, 4])
    with pytest.raises(AssertionError):
        orc.attention(a["q"], a["k"], a["v"], st["cu_seqlens"], st["grids"], text_lens=[-1, 9])
