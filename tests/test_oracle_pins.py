"""Pins for the fp64 oracle (oracle/lspref.py) -- CPU only.

The paper prints no worked numeric example for this path, so the oracle is pinned to
what the mathematics fixes: brute-force pure-Python loops, closed forms (tests/golden/*.txt, derived by
hand), invariants, central finite differences, and independent torch float64 library routines.  Each
test is chosen so that a plausible mistake (dropped term, wrong sign/index, transposed operand, wrong
head mapping, off-by-one in the causal mask) fails at least one of them.
"""
import math
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F
from scipy.special import logsumexp

from oracle import lspref as R

GOLD = os.path.join(os.path.dirname(__file__), "golden")
rng = np.random.default_rng(1234)


def small_cfg(**kw):
    base = dict(batch=2, seq=12, hidden=16, n_q_heads=4, n_kv_heads=2, head_dim=4, ffn=24,
                rms_eps=1e-5, rope_base=10000.0)
    base.update(kw)
    return R.LayerShape(**base)


def rand_weights(cfg, scale=0.3, seed=7):
    g = np.random.default_rng(seed)
    H, Fd, nqd, nkvd = cfg.hidden, cfg.ffn, cfg.nq_dim, cfg.nkv_dim
    return dict(wq=g.normal(0, scale, (nqd, H)), wk=g.normal(0, scale, (nkvd, H)), wv=g.normal(0, scale, (nkvd, H)),
                wo=g.normal(0, scale, (H, nqd)), w_gate=g.normal(0, scale, (Fd, H)), w_up=g.normal(0, scale, (Fd, H)),
                w_down=g.normal(0, scale, (H, Fd)), g_attn=1 + 0.1 * g.normal(size=H), g_mlp=1 + 0.1 * g.normal(size=H))


# ------------------------------------------------------------------------------------------- attention fwd
def brute_attention(q, k, v):
    """Second, deliberately different path: scalar Python loops, full SxS with -inf mask, two-pass softmax."""
    B, S, nq, d = q.shape
    G = nq // k.shape[2]
    O = np.zeros_like(q)
    L = np.zeros((B, nq, S))
    for b in range(B):
        for h in range(nq):
            for i in range(S):
                logits = []
                for j in range(S):
                    if j > i:
                        logits.append(-math.inf)
                    else:
                        logits.append(sum(q[b, i, h, c] * k[b, j, h // G, c] for c in range(d)) / math.sqrt(d))
                den = sum(math.exp(l) for l in logits)
                L[b, h, i] = math.log(den)
                for j in range(S):
                    p = math.exp(logits[j]) / den
                    for c in range(d):
                        O[b, i, h, c] += p * v[b, j, h // G, c]
    return O, L


def test_sdpa_fwd_brute_force():
    q = rng.normal(size=(2, 7, 4, 3)); k = rng.normal(size=(2, 7, 2, 3)); v = rng.normal(size=(2, 7, 2, 3))
    O, L = R.sdpa_fwd(q, k, v)
    Ob, Lb = brute_attention(q, k, v)
    np.testing.assert_allclose(O, Ob, rtol=0, atol=1e-13)
    np.testing.assert_allclose(L, Lb, rtol=0, atol=1e-13)


def test_sdpa_closed_form_golden():
    """tests/golden/attention_closed_form.txt: logits (0, ln3) -> P = (1/4, 3/4); hand-derived from [23]."""
    rows = [l.split() for l in open(os.path.join(GOLD, "attention_closed_form.txt")) if l.strip() and not l.startswith("#")]
    vals = {r[0]: [float(x) for x in r[1:]] for r in rows}
    d = 4
    q = np.zeros((1, 2, 1, d)); k = np.zeros((1, 2, 1, d)); v = np.zeros((1, 2, 1, d))
    q[0, 1, 0, 0] = 2.0                      # q_1 = (2,0,0,0)
    k[0, 1, 0, 0] = math.log(3.0)            # q_1.k_1/sqrt(4) = ln 3 ; q_1.k_0 = 0
    v[0, 0, 0] = [1, 2, 3, 4]; v[0, 1, 0] = [5, 6, 7, 8]
    O, L = R.sdpa_fwd(q, k, v)
    np.testing.assert_allclose(O[0, 0, 0], vals["O0"], atol=1e-15)
    np.testing.assert_allclose(O[0, 1, 0], vals["O1"], atol=1e-14)
    np.testing.assert_allclose(L[0, 0], [vals["L"][0], math.log(4.0)], atol=1e-14)
    assert abs(vals["L"][1] - math.log(4.0)) < 1e-12


def test_softmax_rows_sum_to_one_and_mask():
    q = rng.normal(size=(9, 5)); k = rng.normal(size=(9, 5))
    P, L = R._probs(q, k, 1 / math.sqrt(5))
    np.testing.assert_allclose(P.sum(1), 1.0, atol=1e-15)
    assert np.all(P[np.triu_indices(9, 1)] == 0.0) and np.all(np.diag(P) > 0)
    s = (q @ k.T) / math.sqrt(5)
    for i in range(9):
        assert abs(L[i] - logsumexp(s[i, : i + 1])) < 1e-13


def test_sdpa_closed_forms():
    B, S, nq, nkv, d = 1, 9, 4, 2, 6
    k = rng.normal(size=(B, S, nkv, d)); v = rng.normal(size=(B, S, nkv, d))
    O, L = R.sdpa_fwd(np.zeros((B, S, nq, d)), k, v)            # q = 0  =>  uniform over j <= i
    for h in range(nq):
        run = np.cumsum(v[0, :, h // 2], axis=0) / np.arange(1, S + 1)[:, None]
        np.testing.assert_allclose(O[0, :, h], run, atol=1e-14)
        np.testing.assert_allclose(L[0, h], np.log(np.arange(1, S + 1)), atol=1e-14)
    q1 = rng.normal(size=(3, 1, nq, d)); k1 = rng.normal(size=(3, 1, nkv, d)); v1 = rng.normal(size=(3, 1, nkv, d))
    O1, _ = R.sdpa_fwd(q1, k1, v1)                              # S = 1  =>  O = v of the mapped kv head
    for h in range(nq):
        np.testing.assert_array_equal(O1[:, 0, h], v1[:, 0, h // 2])


def test_sdpa_vs_torch_library():
    B, S, nq, nkv, d = 2, 33, 6, 2, 8
    q = rng.normal(size=(B, S, nq, d)); k = rng.normal(size=(B, S, nkv, d)); v = rng.normal(size=(B, S, nkv, d))
    dO = rng.normal(size=(B, S, nq, d))
    tq, tk, tv = (torch.tensor(t).permute(0, 2, 1, 3).requires_grad_(True) for t in (q, k, v))
    to = F.scaled_dot_product_attention(tq, tk, tv, is_causal=True, enable_gqa=True)
    to.backward(torch.tensor(dO).permute(0, 2, 1, 3))
    O, _ = R.sdpa_fwd(q, k, v)
    dq, dk, dv = R.sdpa_bwd(q, k, v, dO)
    np.testing.assert_allclose(O, to.detach().permute(0, 2, 1, 3).numpy(), atol=1e-12)
    for got, t in ((dq, tq), (dk, tk), (dv, tv)):
        np.testing.assert_allclose(got, t.grad.permute(0, 2, 1, 3).numpy(), atol=1e-12)


def test_packed_sequences_equal_block_diagonal_mask():
    """The reference the packed-sequence GPU tests build (the oracle run on every sequence by itself, results laid end to
    end) is attention over the packed row under a block-diagonal causal mask: checked against torch's float64
    scaled_dot_product_attention with that mask, forward and backward."""
    cu = [0, 5, 6, 19, 33]
    S, nq, nkv, d = cu[-1], 4, 2, 8
    q = rng.normal(size=(1, S, nq, d)); k = rng.normal(size=(1, S, nkv, d)); v = rng.normal(size=(1, S, nkv, d))
    dO = rng.normal(size=(1, S, nq, d))
    start = np.zeros(S, dtype=np.int64)
    for a, b in zip(cu, cu[1:]):
        start[a:b] = a
    idx = np.arange(S)
    mask = torch.tensor((idx[None, :] <= idx[:, None]) & (idx[None, :] >= start[:, None]))      # [query, key]
    tq, tk, tv = (torch.tensor(t).permute(0, 2, 1, 3).requires_grad_(True) for t in (q, k, v))
    to = F.scaled_dot_product_attention(tq, tk, tv, attn_mask=mask, enable_gqa=True)
    to.backward(torch.tensor(dO).permute(0, 2, 1, 3))
    O = np.zeros_like(q); dq = np.zeros_like(q); dk = np.zeros_like(k); dv = np.zeros_like(v)
    for a, b in zip(cu, cu[1:]):
        O[:, a:b], _ = R.sdpa_fwd(q[:, a:b], k[:, a:b], v[:, a:b])
        dq[:, a:b], dk[:, a:b], dv[:, a:b] = R.sdpa_bwd(q[:, a:b], k[:, a:b], v[:, a:b], dO[:, a:b])
    np.testing.assert_allclose(O, to.detach().permute(0, 2, 1, 3).numpy(), atol=1e-12)
    for got, t in ((dq, tq), (dk, tk), (dv, tv)):
        np.testing.assert_allclose(got, t.grad.permute(0, 2, 1, 3).numpy(), atol=1e-12)


def test_gqa_reduces_to_mha_and_group_sum():
    B, S, nq, nkv, d = 1, 10, 6, 2, 4
    G = nq // nkv
    q = rng.normal(size=(B, S, nq, d)); k = rng.normal(size=(B, S, nkv, d)); v = rng.normal(size=(B, S, nkv, d))
    dO = rng.normal(size=(B, S, nq, d))
    kr, vr = np.repeat(k, G, axis=2), np.repeat(v, G, axis=2)    # contiguous groups: head h <- kv h//G
    O, L = R.sdpa_fwd(q, k, v)
    Om, Lm = R.sdpa_fwd(q, kr, vr)                               # nkv == nq : plain MHA
    np.testing.assert_allclose(O, Om, atol=1e-14); np.testing.assert_allclose(L, Lm, atol=1e-14)
    dq, dk, dv = R.sdpa_bwd(q, k, v, dO)
    dqm, dkm, dvm = R.sdpa_bwd(q, kr, vr, dO)
    np.testing.assert_allclose(dq, dqm, atol=1e-13)
    np.testing.assert_allclose(dk, dkm.reshape(B, S, nkv, G, d).sum(3), atol=1e-13)
    np.testing.assert_allclose(dv, dvm.reshape(B, S, nkv, G, d).sum(3), atol=1e-13)
    # MHA special case against an independent single-head loop
    for h in range(nq):
        Oh, _ = R.sdpa_fwd(q[:, :, h:h + 1], kr[:, :, h:h + 1], vr[:, :, h:h + 1])
        np.testing.assert_allclose(Oh[:, :, 0], Om[:, :, h], atol=1e-14)


def test_attention_bwd_identities():
    B, S, nq, nkv, d = 1, 11, 2, 1, 5
    q = rng.normal(size=(B, S, nq, d)); k = rng.normal(size=(B, S, nkv, d)); v = rng.normal(size=(B, S, nkv, d))
    dO = rng.normal(size=(B, S, nq, d))
    O, _ = R.sdpa_fwd(q, k, v)
    dq, dk, dv = R.sdpa_bwd(q, k, v, dO)
    # the identity a flash backward relies on: sum_j P_ij dP_ij == sum_c dO_ic O_ic ; alt path via D
    scale = 1 / math.sqrt(d)
    dq2 = np.zeros_like(dq); dk2 = np.zeros_like(dk)
    for h in range(nq):
        P, _ = R._probs(q[0, :, h], k[0, :, 0], scale)
        dP = dO[0, :, h] @ v[0, :, 0].T
        D = np.sum(dO[0, :, h] * O[0, :, h], axis=1)
        np.testing.assert_allclose(np.sum(P * dP, 1), D, atol=1e-13)
        dS = P * (dP - D[:, None])
        np.testing.assert_allclose(dS.sum(1), 0, atol=1e-13)     # rows of dS sum to zero
        dq2[0, :, h] = dS @ k[0, :, 0] * scale
        dk2[0, :, 0] += dS.T @ q[0, :, h] * scale
    np.testing.assert_allclose(dq, dq2, atol=1e-13); np.testing.assert_allclose(dk, dk2, atol=1e-13)
    # logits shift invariance: adding a constant vector c to every key leaves P unchanged only through q.c,
    # which is constant along j -> O unchanged
    c = rng.normal(size=d)
    O2, _ = R.sdpa_fwd(q, k + c, v)
    np.testing.assert_allclose(O, O2, atol=1e-12)


# ------------------------------------------------------------------------------------------- RoPE
@pytest.mark.parametrize("layout", [0, 1])
def test_rope_properties(layout):
    B, S, nh, d = 2, 9, 3, 8
    z = rng.normal(size=(B, S, nh, d))
    th = R.rope_angles(S, d, 10000.0)
    r = R.rope_apply(z, th, layout)
    pair = (lambda t: t[..., 0::2] ** 2 + t[..., 1::2] ** 2) if layout == 0 else (lambda t: t[..., :d // 2] ** 2 + t[..., d // 2:] ** 2)
    np.testing.assert_allclose(pair(r), pair(z), rtol=1e-14)                      # per-pair norm preserved
    np.testing.assert_array_equal(r[:, 0], z[:, 0])                               # position 0 is the identity
    np.testing.assert_allclose(R.rope_apply(r, th, layout, inverse=True), z, atol=1e-14)   # theta then -theta
    # inverse is the transpose (the backward): <R z, w> == <z, R^T w>
    w = rng.normal(size=z.shape)
    assert abs(np.sum(r * w) - np.sum(z * R.rope_apply(w, th, layout, inverse=True))) < 1e-12


def test_rope_closed_form_and_frequencies():
    d, base = 4, 10000.0
    th = R.rope_angles(5, d, base)
    np.testing.assert_allclose(th[:, 0], np.arange(5), atol=0)                    # i=0: theta = p
    np.testing.assert_allclose(th[:, 1], np.arange(5) * base ** (-2 / d), rtol=1e-15)
    z = np.zeros((1, 5, 1, d)); z[..., 0] = 1.0                                  # (1,0) pair
    r = R.rope_apply(z, th, 0)
    np.testing.assert_allclose(r[0, :, 0, 0], np.cos(np.arange(5)), atol=1e-15)
    np.testing.assert_allclose(r[0, :, 0, 1], np.sin(np.arange(5)), atol=1e-15)   # counter-clockwise by +theta


def test_half_split_rope_is_adjacent_rope_on_interleaved_rows():
    """The identity the library's rope_layout = 1 rests on: with the features of a head
    interleaved, z'[2i] = z[i], z'[2i + 1] = z[i + d/2], adjacent-pair rotation of z' is the interleaved half-split
    rotation of z, and q'.k' = q.k because the same permutation acts on both."""
    S_, h, d = 7, 3, 16
    z = rng.normal(size=(1, S_, h, d)); k = rng.normal(size=(1, S_, h, d))
    th = R.rope_angles(S_, d, 10000.0)
    perm = np.empty(d, dtype=np.int64)
    perm[0::2] = np.arange(d // 2); perm[1::2] = np.arange(d // 2) + d // 2
    np.testing.assert_allclose(R.rope_apply(z[..., perm], th, 0), R.rope_apply(z, th, 1)[..., perm], atol=1e-14)
    a, b = R.rope_apply(z[..., perm], th, 0), R.rope_apply(k[..., perm], th, 0)
    a1, b1 = R.rope_apply(z, th, 1), R.rope_apply(k, th, 1)
    np.testing.assert_allclose(np.einsum("bshd,bthd->bhst", a, b), np.einsum("bshd,bthd->bhst", a1, b1), atol=1e-12)


def test_rope_relative_position_property():
    cfg = small_cfg(batch=1, seq=10)
    w = rand_weights(cfg)
    x = rng.normal(size=(cfg.tokens, cfg.hidden))
    a0, _ = R.attn_block_fwd(x, w, cfg, pos0=0)
    a7, _ = R.attn_block_fwd(x, w, cfg, pos0=7)
    np.testing.assert_allclose(a0, a7, atol=1e-12)      # shifting all positions leaves every q_i.k_j unchanged
    cfg_nr = R.LayerShape(**{**cfg.__dict__, "use_rope": False})
    an, _ = R.attn_block_fwd(x, w, cfg_nr)
    assert np.max(np.abs(an - a0)) > 1e-3               # and RoPE does change the result


# ------------------------------------------------------------------------------------------- RMSNorm / SwiGLU
def test_rmsnorm_pins():
    T, H, eps = 5, 12, 1e-5
    x = rng.normal(size=(T, H)); g = 1 + 0.1 * rng.normal(size=H)
    xn, r = R.rmsnorm_fwd(x, g, eps)
    ms = np.mean(x * x, 1)
    np.testing.assert_allclose(np.mean((xn / g) ** 2, 1), ms / (ms + eps), rtol=1e-13)
    np.testing.assert_allclose(xn, F.rms_norm(torch.tensor(x), (H,), torch.tensor(g), eps).numpy(), atol=1e-14)
    xs, _ = R.rmsnorm_fwd(3.7 * x, g, 0.0); x0, _ = R.rmsnorm_fwd(x, g, 0.0)
    np.testing.assert_allclose(xs, x0, atol=1e-13)                                 # scale invariance at eps = 0
    dxn = rng.normal(size=(T, H))
    dx, dg = R.rmsnorm_bwd(x, g, r, dxn)
    n = x * r[:, None]; dn = dxn * g
    np.testing.assert_allclose(np.sum(dx * x, 1), eps * r ** 2 * np.sum(dn * n, 1), atol=1e-13)
    tx = torch.tensor(x, requires_grad=True); tg = torch.tensor(g, requires_grad=True)
    F.rms_norm(tx, (H,), tg, eps).backward(torch.tensor(dxn))
    np.testing.assert_allclose(dx, tx.grad.numpy(), atol=1e-13); np.testing.assert_allclose(dg, tg.grad.numpy(), atol=1e-13)


def test_swiglu_pins():
    assert R.swiglu_fwd(np.array([0.0]), np.array([3.0]))[0] == 0.0               # silu(0) = 0
    dg, du = R.swiglu_bwd(np.array([0.0]), np.array([3.0]), np.array([2.0]))
    assert dg[0] == 2.0 * 3.0 * 0.5 and du[0] == 0.0                              # silu'(0) = 1/2
    big = R.swiglu_fwd(np.array([40.0]), np.array([1.5]))
    assert abs(big[0] - 60.0) < 1e-12                                             # silu(g) -> g for g >> 0
    g = rng.normal(size=(4, 9)); u = rng.normal(size=(4, 9)); dh = rng.normal(size=(4, 9))
    np.testing.assert_allclose(R.swiglu_fwd(g, u), (F.silu(torch.tensor(g)) * torch.tensor(u)).numpy(), atol=1e-15)
    tg = torch.tensor(g, requires_grad=True); tu = torch.tensor(u, requires_grad=True)
    (F.silu(tg) * tu).backward(torch.tensor(dh))
    dg, du = R.swiglu_bwd(g, u, dh)
    np.testing.assert_allclose(dg, tg.grad.numpy(), atol=1e-14); np.testing.assert_allclose(du, tu.grad.numpy(), atol=1e-14)


def test_linear_orientation():
    """[out,in] weights: a transposed operand anywhere fails this (non-square shapes, hand loops)."""
    x = rng.normal(size=(3, 5)); w = rng.normal(size=(4, 5)); dy = rng.normal(size=(3, 4))
    y = R.linear(x, w)
    for t in range(3):
        for o in range(4):
            assert abs(y[t, o] - sum(x[t, i] * w[o, i] for i in range(5))) < 1e-14
    dx, dw = R.linear_dgrad(dy, w), R.linear_wgrad(dy, x)
    assert dx.shape == x.shape and dw.shape == w.shape
    for t in range(3):
        for i in range(5):
            assert abs(dx[t, i] - sum(dy[t, o] * w[o, i] for o in range(4))) < 1e-14
    for o in range(4):
        for i in range(5):
            assert abs(dw[o, i] - sum(dy[t, o] * x[t, i] for t in range(3))) < 1e-14


# ------------------------------------------------------------------------------------------- whole layer
def test_causality_bit_identical():
    cfg = small_cfg(batch=2, seq=9)
    w = rand_weights(cfg)
    x = rng.normal(size=(cfg.tokens, cfg.hidden))
    y, _ = R.layer_fwd(x, w, cfg)
    t = 4
    x2 = x.copy()
    for b in range(cfg.batch):
        x2[b * cfg.seq + t + 1: (b + 1) * cfg.seq] += rng.normal(size=(cfg.seq - t - 1, cfg.hidden))
    y2, _ = R.layer_fwd(x2, w, cfg)
    for b in range(cfg.batch):
        s = slice(b * cfg.seq, b * cfg.seq + t + 1)
        np.testing.assert_allclose(y[s], y2[s], rtol=0, atol=1e-13)
        assert np.max(np.abs(y[b * cfg.seq + t + 1:(b + 1) * cfg.seq] - y2[b * cfg.seq + t + 1:(b + 1) * cfg.seq])) > 1e-3
    # sequences in a batch are independent: changing batch 1 leaves batch 0 untouched
    x3 = x.copy(); x3[cfg.seq:] += 1.0
    y3, _ = R.layer_fwd(x3, w, cfg)
    np.testing.assert_allclose(y[:cfg.seq], y3[:cfg.seq], rtol=0, atol=1e-13)


def test_zero_branch_weights():
    cfg = small_cfg()
    w = rand_weights(cfg); w["wo"] = np.zeros_like(w["wo"]); w["w_down"] = np.zeros_like(w["w_down"])
    x = rng.normal(size=(cfg.tokens, cfg.hidden)); dy = rng.normal(size=(cfg.tokens, cfg.hidden))
    out = R.layer_fwd_bwd(x, dy, w, cfg)
    np.testing.assert_array_equal(out["y"], x); np.testing.assert_array_equal(out["dx"], dy)
    for kname in ("dwq", "dwk", "dwv", "dw_gate", "dw_up", "dg_attn", "dg_mlp"):
        assert not np.any(out[kname]), kname
    assert np.any(out["dwo"]) and np.any(out["dw_down"])


def test_block_composition_and_linearity():
    cfg = small_cfg()
    w = rand_weights(cfg)
    x = rng.normal(size=(cfg.tokens, cfg.hidden)); dy = rng.normal(size=(cfg.tokens, cfg.hidden))
    out = R.layer_fwd_bwd(x, dy, w, cfg)
    a, ca = R.attn_block_fwd(x, w, cfg); y, cm = R.mlp_block_fwd(a, w, cfg)
    np.testing.assert_array_equal(out["y"], y)
    da, gm = R.mlp_block_bwd(dy, w, cfg, cm); dx, ga = R.attn_block_bwd(da, w, cfg, ca)
    np.testing.assert_array_equal(out["dx"], dx); np.testing.assert_array_equal(out["da"], da)
    w2 = dict(w); w2["w_down"] = 2.5 * w["w_down"]
    y2, _ = R.mlp_block_fwd(a, w2, cfg)
    np.testing.assert_allclose(y2 - a, 2.5 * (y - a), atol=1e-12)                 # y - a linear in Wd


def loss(x, dy, w, cfg):
    y, _ = R.layer_fwd(x, w, cfg)
    return float(np.sum(y * dy))


@pytest.mark.parametrize("rope_layout", [0, 1])
def test_finite_difference_all_gradients(rope_layout):
    cfg = small_cfg(batch=2, seq=6, hidden=8, n_q_heads=4, n_kv_heads=2, head_dim=4, ffn=12, rope_layout=rope_layout)
    w = rand_weights(cfg, scale=0.4)
    g = np.random.default_rng(99)
    x = g.normal(size=(cfg.tokens, cfg.hidden)); dy = g.normal(size=(cfg.tokens, cfg.hidden))
    out = R.layer_fwd_bwd(x, dy, w, cfg)
    eps = 1e-6
    for name in ("x",) + tuple(w.keys()):
        base = x if name == "x" else w[name]
        grad = out["dx"] if name == "x" else out["d" + name]
        assert grad.shape == base.shape
        for trial in range(3):
            delta = g.normal(size=base.shape); delta /= np.linalg.norm(delta)
            def at(s):
                if name == "x":
                    return loss(x + s * delta, dy, w, cfg)
                w2 = dict(w); w2[name] = base + s * delta
                return loss(x, dy, w2, cfg)
            fd = (at(eps) - at(-eps)) / (2 * eps)
            an = float(np.sum(grad * delta))
            assert abs(fd - an) <= 2e-7 * max(1.0, abs(an)), (name, trial, fd, an)


def torch_layer(x, w, cfg):
    """Independent composite written HF-style in torch float64 (half-split RoPE on permuted weights is
    avoided: uses complex multiplication for adjacent pairs), autograd for gradients."""
    B, S, nq, nkv, d = cfg.batch, cfg.seq, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    def norm(t, g):
        return t * torch.rsqrt(t.pow(2).mean(-1, keepdim=True) + cfg.rms_eps) * g
    xn = norm(x, w["g_attn"])
    q = (xn @ w["wq"].T).view(B, S, nq, d); k = (xn @ w["wk"].T).view(B, S, nkv, d); v = (xn @ w["wv"].T).view(B, S, nkv, d)
    freqs = torch.outer(torch.arange(S, dtype=torch.float64),
                        cfg.rope_base ** (-torch.arange(0, d, 2, dtype=torch.float64) / d))
    cis = torch.polar(torch.ones_like(freqs), freqs)[None, :, None, :]
    rot = lambda t: torch.view_as_real(torch.view_as_complex(t.reshape(*t.shape[:-1], d // 2, 2)) * cis).flatten(3)
    q, k = rot(q), rot(k)
    o = F.scaled_dot_product_attention(q.transpose(1, 2), k.transpose(1, 2), v.transpose(1, 2), is_causal=True, enable_gqa=True)
    a = x + o.transpose(1, 2).reshape(B * S, nq * d) @ w["wo"].T
    an = norm(a, w["g_mlp"])
    return a + (F.silu(an @ w["w_gate"].T) * (an @ w["w_up"].T)) @ w["w_down"].T


def test_layer_vs_torch_autograd():
    cfg = small_cfg(batch=2, seq=17, hidden=24, n_q_heads=6, n_kv_heads=2, head_dim=8, ffn=40)
    w = rand_weights(cfg)
    x = rng.normal(size=(cfg.tokens, cfg.hidden)); dy = rng.normal(size=(cfg.tokens, cfg.hidden))
    out = R.layer_fwd_bwd(x, dy, w, cfg)
    tw = {k: torch.tensor(v, requires_grad=True) for k, v in w.items()}
    tx = torch.tensor(x, requires_grad=True)
    ty = torch_layer(tx, tw, cfg)
    ty.backward(torch.tensor(dy))
    np.testing.assert_allclose(out["y"], ty.detach().numpy(), atol=1e-12)
    np.testing.assert_allclose(out["dx"], tx.grad.numpy(), atol=1e-11)
    for k in w:
        np.testing.assert_allclose(out["d" + k], tw[k].grad.numpy(), atol=1e-11, err_msg=k)


def test_embed_and_stack():
    table = rng.normal(size=(11, 6)); ids = np.array([3, 0, 10, 3], np.int32)
    x0 = R.embed_fwd(ids, table)
    for t, i in enumerate(ids):
        np.testing.assert_array_equal(x0[t], table[i])
    cfg = small_cfg(batch=1, seq=4, hidden=6, n_q_heads=2, n_kv_heads=1, head_dim=4, ffn=10)
    ws = [rand_weights(cfg, seed=s) for s in (1, 2, 3)]
    dy = rng.normal(size=(4, 6))
    y, dx0, grads = R.stack_fwd_bwd(x0, dy, ws, cfg)
    xs = x0
    caches = []
    for w in ws:
        xs, c = R.layer_fwd(xs, w, cfg); caches.append(c)
    np.testing.assert_array_equal(y, xs)
    d = dy
    for li in (2, 1, 0):
        d, g, _ = R.layer_bwd(d, ws[li], cfg, caches[li])
        for k in g:
            np.testing.assert_array_equal(g[k], grads[li][k])
    np.testing.assert_array_equal(d, dx0)
