"""emulate16 -- the oracle's EMULATION mode: the same layer forward + backward as lspref.py, in float64, with the values
rounded to 16 bits at exactly the places where a tensor-core implementation has to feed 16-bit operands
(precision plan and Appendix B).

TEST INFRASTRUCTURE ONLY, same rules as lspref.py (only tests/ and the scripts under tests/golden/ import it; it shares
no code with the CUDA path).  It is NOT a second oracle: parity is always judged against lspref.py.  Its one use is
the "emulated-precision floor" SURVEY 8(c) asks to report beside a GPU error that exceeds the 2e-2 bar: the error a
CORRECT implementation with 16-bit operands and exact (here float64) accumulation makes against the exact definition.
If the CUDA path sits at this floor, the excess is the price of the operand format, not a defect of the kernels.

Rounding sites (fmt = "f16": IEEE half, the CUDA path's operand format, P-2'; "bf16": the paper's BF16,
PAPER.md:73), everything else exact:
  forward : xn, an (normalised activations) | q, k (after RoPE), v | P (relative to the row maximum) | O as the
            O-projection operand (the saved fp32 O stays exact, P-3) | h = silu(g) u | the saved g, u
  backward: dy, da as GEMM operands | dg, du | dO | P and dS (exact for query positions < split_rows: the hi + lo
            split of P-5 / P-6) | dq, dk (after the inverse rotation), dv
Weights are bf16 values: exact in either format for |w| in the normal range.
"""
from __future__ import annotations

import math

import numpy as np

from . import lspref as R

F64 = np.float64


def make_rounder(fmt: str):
    if fmt == "exact":                       # no rounding at all: the emulation must then BE lspref (pinned in the tests)
        return lambda a: np.asarray(a, F64)
    if fmt == "f16":
        return lambda a: np.asarray(a, F64).astype(np.float16).astype(F64)
    if fmt == "bf16":
        def r(a):
            u = np.ascontiguousarray(np.asarray(a, np.float32)).view(np.uint32)
            u = (u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))) & np.uint32(0xFFFF0000)
            return u.view(np.float32).astype(F64)
        return r
    raise ValueError(fmt)


def layer_fwd(x, w, cfg: R.LayerShape, rnd):
    """Forward of one layer with 16-bit operands.  Returns (y, cache)."""
    B, S, nq, nkv, d = cfg.batch, cfg.seq, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    G = nq // nkv
    x = np.asarray(x, F64)
    xn_exact, r1 = R.rmsnorm_fwd(x, w["g_attn"], cfg.rms_eps)
    xn = rnd(xn_exact)
    q = R.linear(xn, w["wq"]).reshape(B, S, nq, d)
    k = R.linear(xn, w["wk"]).reshape(B, S, nkv, d)
    v = R.linear(xn, w["wv"]).reshape(B, S, nkv, d)
    theta = R.rope_angles(S, d, cfg.rope_base) if cfg.use_rope else None
    if cfg.use_rope:
        q = R.rope_apply(q, theta, cfg.rope_layout)
        k = R.rope_apply(k, theta, cfg.rope_layout)
    q, k, v = rnd(q), rnd(k), rnd(v)
    scale = 1.0 / math.sqrt(d)
    O = np.empty_like(q)
    L = np.empty((B, nq, S), F64)
    for b in range(B):
        for h in range(nq):
            s = np.matmul(q[b, :, h], k[b, :, h // G].T) * scale
            s[np.triu_indices(S, k=1)] = -np.inf
            m = np.max(s, axis=1)
            e = np.exp(s - m[:, None])
            z = np.sum(e, axis=1)                                  # row sums of the unrounded exponentials (fp32 on the GPU)
            O[b, :, h] = np.matmul(rnd(e), v[b, :, h // G]) / z[:, None]
            L[b, h] = m + np.log(z)
    O2 = O.reshape(B * S, nq * d)
    a = x + R.linear(rnd(O2), w["wo"])
    an_exact, r2 = R.rmsnorm_fwd(a, w["g_mlp"], cfg.rms_eps)
    an = rnd(an_exact)
    g = R.linear(an, w["w_gate"])
    u = R.linear(an, w["w_up"])
    h_ = rnd(R.swiglu_fwd(g, u))
    y = a + R.linear(h_, w["w_down"])
    return y, dict(x=x, xn=xn, r1=r1, q=q, k=k, v=v, O=O2, L=L, theta=theta, a=a, an=an, r2=r2, g=rnd(g), u=rnd(u), h=h_)


def layer_bwd(dy, w, cfg: R.LayerShape, c, rnd, split_rows=256):
    """Backward of one layer with 16-bit operands.  Returns (dx, grads)."""
    B, S, nq, nkv, d = cfg.batch, cfg.seq, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    G = nq // nkv
    T = B * S
    dy = np.asarray(dy, F64)
    dy16 = rnd(dy)
    grads = {}
    # MLP block
    grads["w_down"] = R.linear_wgrad(dy16, c["h"])
    dh = R.linear_dgrad(dy16, w["w_down"])
    dg, du = R.swiglu_bwd(c["g"], c["u"], dh)
    dg, du = rnd(dg), rnd(du)
    grads["w_gate"] = R.linear_wgrad(dg, c["an"])
    grads["w_up"] = R.linear_wgrad(du, c["an"])
    dan = R.linear_dgrad(dg, w["w_gate"]) + R.linear_dgrad(du, w["w_up"])
    da_n, grads["g_mlp"] = R.rmsnorm_bwd(c["a"], w["g_mlp"], c["r2"], dan)
    da = dy + da_n
    da16 = rnd(da)
    # attention block
    O16 = rnd(c["O"])
    grads["wo"] = R.linear_wgrad(da16, O16)
    dO = rnd(R.linear_dgrad(da16, w["wo"]))
    dO4 = dO.reshape(B, S, nq, d)
    O4 = c["O"].reshape(B, S, nq, d)
    q, k, v = c["q"], c["k"], c["v"]
    scale = 1.0 / math.sqrt(d)
    dq = np.zeros_like(q); dk = np.zeros_like(k); dv = np.zeros_like(v)
    early = np.arange(S) < split_rows                               # query positions whose P / dS keep hi + lo halves
    for b in range(B):
        for h in range(nq):
            kv = h // G
            s = np.matmul(q[b, :, h], k[b, :, kv].T) * scale
            s[np.triu_indices(S, k=1)] = -np.inf
            P = np.exp(s - c["L"][b, h][:, None])                   # recomputed from the saved log-sum-exp
            P16 = rnd(P)
            P16[early] = P[early]
            dv[b, :, kv] += np.matmul(P16.T, dO4[b, :, h])
            dP = np.matmul(dO4[b, :, h], v[b, :, kv].T)
            D = np.sum(dO4[b, :, h] * O4[b, :, h], axis=1)          # rowsum(dO * O) with the exact (fp32) O
            dS = P * (dP - D[:, None])
            dS16 = rnd(dS)
            dS16[early] = dS[early]
            dq[b, :, h] = np.matmul(dS16, k[b, :, kv]) * scale
            dk[b, :, kv] += np.matmul(dS16.T, q[b, :, h]) * scale
    if cfg.use_rope:
        dq = R.rope_apply(dq, c["theta"], cfg.rope_layout, inverse=True)
        dk = R.rope_apply(dk, c["theta"], cfg.rope_layout, inverse=True)
    dq2, dk2, dv2 = rnd(dq.reshape(T, nq * d)), rnd(dk.reshape(T, nkv * d)), rnd(dv.reshape(T, nkv * d))
    dxn = R.linear_dgrad(dq2, w["wq"]) + R.linear_dgrad(dk2, w["wk"]) + R.linear_dgrad(dv2, w["wv"])
    grads["wq"] = R.linear_wgrad(dq2, c["xn"])
    grads["wk"] = R.linear_wgrad(dk2, c["xn"])
    grads["wv"] = R.linear_wgrad(dv2, c["xn"])
    dx_n, grads["g_attn"] = R.rmsnorm_bwd(c["x"], w["g_attn"], c["r1"], dxn)
    return da + dx_n, grads


def stack_fwd_bwd(x0, dy, weights, cfg: R.LayerShape, fmt="f16", on_layer_grads=None):
    """The stack of lspref.stack_fwd_bwd with 16-bit operands (layer inputs kept, internals recomputed in the backward).
    on_layer_grads(layer, grads): called per layer instead of collecting every gradient.  Returns (y, dx0, grads or None)."""
    rnd = make_rounder(fmt)
    xs = [np.asarray(x0, F64)]
    for w in weights:
        y, _ = layer_fwd(xs[-1], w, cfg, rnd)
        xs.append(y)
    y = xs[-1]
    d = np.asarray(dy, F64)
    all_grads = None if on_layer_grads else [None] * len(weights)
    for li in range(len(weights) - 1, -1, -1):
        wl = weights[li]
        _, cache = layer_fwd(xs[li], wl, cfg, rnd)
        d, grads = layer_bwd(d, wl, cfg, cache, rnd)
        if on_layer_grads:
            on_layer_grads(li, grads)
        else:
            all_grads[li] = grads
    return y, d, all_grads
