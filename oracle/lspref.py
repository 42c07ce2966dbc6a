"""lspref -- the fp64 CPU oracle for the Llama decoder-layer forward+backward.

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this
module.  It shares no code with the CUDA path (``paper_2510_02483_b200/``) and
imports nothing from it; inputs are handed in as numpy arrays.

What it is: the *plain definition* of the standard Llama decoder layer the
paper names (section 2.4: RMSNorm [34], SwiGLU [35], RoPE [36],
GQA [37] / MHA; softmax attention [23]) and its exact gradients
("forward and backward pass operations"), in float64 throughout
(the paper's BF16 mixed precision, only fixes the *storage* type
of the inputs; bf16 -> float64 widening is exact).  No tiling, no online
softmax, no saved-LSE recompute, no fusion: every step is one numpy statement
that can be checked against the formula by eye.  ``numpy.matmul`` (float64) is
the only library primitive used as a step.

The paper gives no equations for these components; the formulas are the ones
of the cited references, in the reading listed in DESIGN.md section 3
(SURVEY.md section 8(c), A-1 .. A-17).  Every function says which.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): brute-force pure-Python
loops on tiny shapes, central finite differences, closed forms, invariants
(softmax rows sum to 1, causality, GQA(nkv=nq)==MHA, RoPE norm/relative
position), and torch float64 library routines as an independent second opinion.
No function here is "parity unpinned" with respect to the mathematics; the
paper itself prints no worked numeric example for this path.

Layouts (row-major numpy):
  x, a, y, dx, da, dy : [T, H]          T = B*S tokens, sequence-major (t = b*S + s)
  wq [Nq,H] wk [Nkv,H] wv [Nkv,H] wo [H,Nq] w_gate [F,H] w_up [F,H] w_down [H,F]   ([out,in])
  g_attn, g_mlp       : [H]
  q [B,S,nq,d]  k,v [B,S,nkv,d]  O [B,S,nq,d]  L [B,nq,S]
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

F64 = np.float64


@dataclass(frozen=True)
class LayerShape:
    """Shape/hyper-parameters of one decoder layer (BASELINE.json configs)."""
    batch: int
    seq: int
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int
    rms_eps: float = 1e-5
    rope_base: float = 10000.0
    rope_layout: int = 0      # 0: adjacent pairs (2i,2i+1) as in [36]; 1: half-split (i, i+d/2)
    use_rope: bool = True

    @property
    def tokens(self) -> int:
        return self.batch * self.seq

    @property
    def nq_dim(self) -> int:
        return self.n_q_heads * self.head_dim

    @property
    def nkv_dim(self) -> int:
        return self.n_kv_heads * self.head_dim


# --------------------------------------------------------------------------- RMSNorm [34]
def rmsnorm_fwd(x, g, eps):
    """RMSNorm (ref [34]; reading A-3: eps inside the sqrt, gain after).

    r_t = 1/sqrt(mean_j x_tj^2 + eps);  xn_tj = x_tj * r_t * g_j.  Returns (xn, r).
    """
    x = np.asarray(x, F64)
    g = np.asarray(g, F64)
    r = 1.0 / np.sqrt(np.mean(x * x, axis=1) + eps)          # [T]
    xn = x * r[:, None] * g[None, :]
    return xn, r


def rmsnorm_bwd(x, g, r, dxn):
    """Exact gradient of rmsnorm_fwd (SURVEY 8(c) backward definition).

    n = x*r, dn = dxn*g;  dx = r*(dn - n*mean_j(dn_j n_j));  dg_j = sum_t dxn_tj n_tj.
    Returns (dx, dg) -- dx is the norm-branch gradient only (no residual term).
    """
    x = np.asarray(x, F64)
    n = x * r[:, None]
    dn = dxn * g[None, :]
    dx = r[:, None] * (dn - n * np.mean(dn * n, axis=1)[:, None])
    dg = np.sum(dxn * n, axis=0)
    return dx, dg


# --------------------------------------------------------------------------- bias-free linear
def linear(x, w):
    """y = x W^T for W stored [out,in] (reading A-2/A-9: no bias)."""
    return np.matmul(x, w.T)


def linear_dgrad(dy, w):
    """dx = dy W."""
    return np.matmul(dy, w)


def linear_wgrad(dy, x):
    """dW = dy^T x  (sum over tokens)."""
    return np.matmul(dy.T, x)


# --------------------------------------------------------------------------- RoPE [36]
def rope_angles(seq, head_dim, base, pos0=0):
    """theta[p, i] = (pos0 + p) * base^(-2i/d), i = 0..d/2-1 (ref [36]; reading A-5: no scaling)."""
    i = np.arange(head_dim // 2, dtype=F64)
    inv_freq = np.power(F64(base), -2.0 * i / head_dim)
    p = np.arange(seq, dtype=F64) + F64(pos0)
    return p[:, None] * inv_freq[None, :]                     # [S, d/2]


def rope_apply(z, theta, layout=0, inverse=False):
    """Rotate every pair of every head of z [B,S,nh,d] by +theta (or -theta if inverse).

    layout 0 (ref [36], reading A-4): pair i = (z[2i], z[2i+1]);
    layout 1: pair i = (z[i], z[i+d/2]).
    (z0, z1) <- (z0 cos - z1 sin, z0 sin + z1 cos).  The inverse rotation is the
    transpose, i.e. the exact backward of the forward rotation.
    """
    z = np.asarray(z, F64)
    d = z.shape[-1]
    c = np.cos(theta)[None, :, None, :]
    s = np.sin(theta)[None, :, None, :]
    if inverse:
        s = -s
    out = np.empty_like(z)
    if layout == 0:
        z0, z1 = z[..., 0::2], z[..., 1::2]
        out[..., 0::2] = z0 * c - z1 * s
        out[..., 1::2] = z0 * s + z1 * c
    else:
        z0, z1 = z[..., : d // 2], z[..., d // 2:]
        out[..., : d // 2] = z0 * c - z1 * s
        out[..., d // 2:] = z0 * s + z1 * c
    return out


# --------------------------------------------------------------------------- causal GQA attention [23],[37]
def _probs(qh, kh, scale):
    """Causal softmax probabilities of one head: P [S,S], and the log-sum-exp L [S].

    s_ij = q_i.k_j * scale for j <= i; entries j > i are excluded (reading A-6:
    the diagonal is included, excluded entries contribute exactly 0).
    """
    S = qh.shape[0]
    s = np.matmul(qh, kh.T) * scale
    s[np.triu_indices(S, k=1)] = -np.inf
    m = np.max(s, axis=1)
    e = np.exp(s - m[:, None])
    z = np.sum(e, axis=1)
    return e / z[:, None], m + np.log(z)


def sdpa_fwd(q, k, v):
    """O_i = sum_{j<=i} softmax_j(q_i.k_j/sqrt(d)) v_j ;  L_i = log sum_{j<=i} exp(q_i.k_j/sqrt(d)).

    q [B,S,nq,d], k,v [B,S,nkv,d]; query head h reads kv head h // (nq/nkv)
    (ref [37], reading A-7).  Returns O [B,S,nq,d], L [B,nq,S].
    """
    q, k, v = (np.asarray(t, F64) for t in (q, k, v))
    B, S, nq, d = q.shape
    G = nq // k.shape[2]
    scale = 1.0 / math.sqrt(d)
    O = np.empty_like(q)
    L = np.empty((B, nq, S), F64)
    for b in range(B):
        for h in range(nq):
            P, L[b, h] = _probs(q[b, :, h], k[b, :, h // G], scale)
            O[b, :, h] = np.matmul(P, v[b, :, h // G])
    return O, L


def sdpa_bwd(q, k, v, dO):
    """Exact gradients of sdpa_fwd from the full P, explicit softmax Jacobian:

    dV_j = sum_h sum_i P_ij dO_i ; dP_ij = dO_i.v_j ; dS_ij = P_ij (dP_ij - sum_j' P_ij' dP_ij') ;
    dq_i = sum_j dS_ij k_j / sqrt(d) ; dk_j = sum_h sum_i dS_ij q_i / sqrt(d); sum_h over the G
    query heads of the kv head.  (The row term is sum_j P dP, *not* rowsum(dO*O).)
    """
    q, k, v, dO = (np.asarray(t, F64) for t in (q, k, v, dO))
    B, S, nq, d = q.shape
    G = nq // k.shape[2]
    scale = 1.0 / math.sqrt(d)
    dq, dk, dv = np.zeros_like(q), np.zeros_like(k), np.zeros_like(v)
    for b in range(B):
        for h in range(nq):
            kv = h // G
            P, _ = _probs(q[b, :, h], k[b, :, kv], scale)
            dv[b, :, kv] += np.matmul(P.T, dO[b, :, h])
            dP = np.matmul(dO[b, :, h], v[b, :, kv].T)
            dS = P * (dP - np.sum(P * dP, axis=1)[:, None])
            dq[b, :, h] = np.matmul(dS, k[b, :, kv]) * scale
            dk[b, :, kv] += np.matmul(dS.T, q[b, :, h]) * scale
    return dq, dk, dv


# --------------------------------------------------------------------------- SwiGLU [35]
def _sigmoid(z):
    return 1.0 / (1.0 + np.exp(-z))


def swiglu_fwd(g, u):
    """h = silu(g) * u, silu(z) = z*sigmoid(z) (ref [35], reading A-8: the gate branch is SiLU'd)."""
    return g * _sigmoid(g) * u


def swiglu_bwd(g, u, dh):
    """du = dh*g*sig(g);  dg = dh*u*sig(g)*(1 + g*(1 - sig(g)))."""
    sg = _sigmoid(g)
    return dh * u * sg * (1.0 + g * (1.0 - sg)), dh * g * sg


# --------------------------------------------------------------------------- attention block
def attn_block_fwd(x, w, cfg: LayerShape, pos0=0):
    """a = x + Wo . GQA(RoPE(Wq xn), RoPE(Wk xn), Wv xn),  xn = RMSNorm(x; g_attn)  (SURVEY 8(c) fwd 1-5).

    w: dict with wq, wk, wv, wo, g_attn.  Returns (a, cache).
    """
    B, S, nq, nkv, d = cfg.batch, cfg.seq, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    x = np.asarray(x, F64)
    xn, r1 = rmsnorm_fwd(x, w["g_attn"], cfg.rms_eps)
    q = linear(xn, w["wq"]).reshape(B, S, nq, d)
    k = linear(xn, w["wk"]).reshape(B, S, nkv, d)
    v = linear(xn, w["wv"]).reshape(B, S, nkv, d)
    theta = rope_angles(S, d, cfg.rope_base, pos0) if cfg.use_rope else None
    if cfg.use_rope:
        q = rope_apply(q, theta, cfg.rope_layout)
        k = rope_apply(k, theta, cfg.rope_layout)
    O, L = sdpa_fwd(q, k, v)
    a = x + linear(O.reshape(B * S, nq * d), w["wo"])
    return a, dict(x=x, xn=xn, r1=r1, q=q, k=k, v=v, O=O, L=L, theta=theta)


def attn_block_bwd(da, w, cfg: LayerShape, c):
    """Exact gradients of attn_block_fwd.  Returns (dx, grads) with wq, wk, wv, wo, g_attn."""
    B, S, nq, nkv, d = cfg.batch, cfg.seq, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim
    T = B * S
    da = np.asarray(da, F64)
    O2 = c["O"].reshape(T, nq * d)
    dwo = linear_wgrad(da, O2)
    dO = linear_dgrad(da, w["wo"]).reshape(B, S, nq, d)
    dq, dk, dv = sdpa_bwd(c["q"], c["k"], c["v"], dO)
    if cfg.use_rope:
        dq = rope_apply(dq, c["theta"], cfg.rope_layout, inverse=True)
        dk = rope_apply(dk, c["theta"], cfg.rope_layout, inverse=True)
    dq2, dk2, dv2 = dq.reshape(T, nq * d), dk.reshape(T, nkv * d), dv.reshape(T, nkv * d)
    dxn = linear_dgrad(dq2, w["wq"]) + linear_dgrad(dk2, w["wk"]) + linear_dgrad(dv2, w["wv"])
    dx_n, dg = rmsnorm_bwd(c["x"], w["g_attn"], c["r1"], dxn)
    grads = dict(wq=linear_wgrad(dq2, c["xn"]), wk=linear_wgrad(dk2, c["xn"]),
                 wv=linear_wgrad(dv2, c["xn"]), wo=dwo, g_attn=dg)
    return da + dx_n, grads


# --------------------------------------------------------------------------- MLP block
def mlp_block_fwd(a, w, cfg: LayerShape):
    """y = a + Wd . (silu(Wg an) * (Wu an)),  an = RMSNorm(a; g_mlp)  (SURVEY 8(c) fwd 6-8)."""
    a = np.asarray(a, F64)
    an, r2 = rmsnorm_fwd(a, w["g_mlp"], cfg.rms_eps)
    g = linear(an, w["w_gate"])
    u = linear(an, w["w_up"])
    h = swiglu_fwd(g, u)
    y = a + linear(h, w["w_down"])
    return y, dict(a=a, an=an, r2=r2, g=g, u=u, h=h)


def mlp_block_bwd(dy, w, cfg: LayerShape, c):
    """Exact gradients of mlp_block_fwd.  Returns (da, grads) with w_gate, w_up, w_down, g_mlp."""
    dy = np.asarray(dy, F64)
    dwd = linear_wgrad(dy, c["h"])
    dh = linear_dgrad(dy, w["w_down"])
    dg, du = swiglu_bwd(c["g"], c["u"], dh)
    dan = linear_dgrad(dg, w["w_gate"]) + linear_dgrad(du, w["w_up"])
    da_n, dgm = rmsnorm_bwd(c["a"], w["g_mlp"], c["r2"], dan)
    grads = dict(w_gate=linear_wgrad(dg, c["an"]), w_up=linear_wgrad(du, c["an"]), w_down=dwd, g_mlp=dgm)
    return dy + da_n, grads


# --------------------------------------------------------------------------- whole layer
def layer_fwd(x, w, cfg: LayerShape):
    """layer = mlp o attn (pre-norm, two residual adds; reading A-2)."""
    a, ca = attn_block_fwd(x, w, cfg)
    y, cm = mlp_block_fwd(a, w, cfg)
    return y, dict(attn=ca, mlp=cm, a=a)


def layer_bwd(dy, w, cfg: LayerShape, cache):
    da, gm = mlp_block_bwd(dy, w, cfg, cache["mlp"])
    dx, ga = attn_block_bwd(da, w, cfg, cache["attn"])
    grads = dict(ga)
    grads.update(gm)
    return dx, grads, da


def layer_fwd_bwd(x, dy, w, cfg: LayerShape):
    """One training step of one layer with loss l = sum(y*dy).  Returns dict of every compared tensor."""
    y, cache = layer_fwd(x, w, cfg)
    dx, grads, da = layer_bwd(dy, w, cfg, cache)
    out = dict(y=y, a=cache["a"], dx=dx, da=da)
    out.update({"d" + k: v for k, v in grads.items()})
    return out


# --------------------------------------------------------------------------- embedding + stack (cfg 3)
def embed_fwd(ids, table):
    """x0[t,:] = E[id_t,:] (BASELINE.json cfg 3; the only integer step on the path)."""
    return np.asarray(table, F64)[np.asarray(ids, np.int64)]


def stack_fwd_bwd(x0, dy, weights, cfg: LayerShape):
    """L decoder layers forward then backward (reading A-11: no final norm/head/loss; dy at the last output).

    weights: list of per-layer dicts.  Keeps only each layer's input and recomputes the layer's
    internals in its backward (memory), which does not change any value.
    Returns (y, dx0, [per-layer grads]).
    """
    xs = [np.asarray(x0, F64)]
    for w in weights:
        y, _ = layer_fwd(xs[-1], w, cfg)
        xs.append(y)
    y = xs[-1]
    d = np.asarray(dy, F64)
    all_grads = [None] * len(weights)
    for li in range(len(weights) - 1, -1, -1):
        _, cache = layer_fwd(xs[li], weights[li], cfg)
        d, grads, _ = layer_bwd(d, weights[li], cfg, cache)
        all_grads[li] = grads
    return y, d, all_grads
