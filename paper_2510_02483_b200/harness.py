"""Device-side plumbing shared by tests/ and bench.py: upload seeded inputs, allocate the caller-owned
buffers of include/lsp.h with torch, call the binding, download results.  No arithmetic of the method
lives here and nothing here imports the oracle.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as B
from . import synth

WEIGHT_SHAPES = lambda w: dict(  # noqa: E731
    wq=(w.n_q_heads * w.head_dim, w.hidden), wk=(w.n_kv_heads * w.head_dim, w.hidden),
    wv=(w.n_kv_heads * w.head_dim, w.hidden), wo=(w.hidden, w.n_q_heads * w.head_dim), g_attn=(w.hidden,),
    w_gate=(w.ffn, w.hidden), w_up=(w.ffn, w.hidden), w_down=(w.hidden, w.ffn), g_mlp=(w.hidden,))


def require_cuda():
    if not torch.cuda.is_available():
        raise B.LspError("no CUDA device: the product path has no CPU fallback")
    return torch.device("cuda", torch.cuda.current_device())


def bf16_to_device(bits: np.ndarray, dev=None) -> torch.Tensor:
    """uint16 bf16 bit patterns -> torch.bfloat16 tensor on the device (bit-exact)."""
    dev = dev or require_cuda()
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(dev)
    return t.view(torch.bfloat16)


def bf16_pinned(bits: np.ndarray) -> torch.Tensor:
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    return t.pin_memory()


def make_ctx(w: synth.Workload, use_rope=True, in_dtype=B.LSP_BF16, **desc_kw) -> B.Ctx:
    """desc_kw: rope_layout (0 / 1), wgrad_accumulate (bool)."""
    return B.Ctx(batch=w.batch, seq=w.seq, hidden=w.hidden, n_q_heads=w.n_q_heads, n_kv_heads=w.n_kv_heads,
                 head_dim=w.head_dim, ffn=w.ffn, rms_eps=w.rms_eps, rope_base=w.rope_base, use_rope=use_rope,
                 in_dtype=in_dtype, device=torch.cuda.current_device(), **desc_kw)


class LayerBuffers:
    """All caller-owned device buffers of one layer shape: saved, ws, outputs and the nine gradients."""

    def __init__(self, ctx: B.Ctx, w: synth.Workload, dev=None):
        dev = dev or require_cuda()
        self.dev = dev
        T, H = w.tokens, w.hidden
        self.saved = torch.empty(ctx.saved_bytes, dtype=torch.uint8, device=dev)
        self.ws = torch.empty(ctx.workspace_bytes, dtype=torch.uint8, device=dev)
        self.y = torch.empty((T, H), dtype=torch.float32, device=dev)
        self.dx = torch.empty((T, H), dtype=torch.float32, device=dev)
        self.grads = {k: torch.empty(s, dtype=torch.float32, device=dev) for k, s in WEIGHT_SHAPES(w).items()}


def upload_weights(wbits: dict, dev=None) -> dict:
    return {k: bf16_to_device(v, dev) for k, v in wbits.items()}


def with_weight_cache(ctx: B.Ctx, weights: dict, dev=None, stream=None) -> dict:
    """The same weight dict plus "f16_cache": the fp16 operand copies of the seven projection weights, converted once by
    lsp_layer_prepare_weights (include/lsp.h: lsp_layer_weights.f16_cache).  Valid until the bf16 weights change."""
    dev = dev or require_cuda()
    cache = torch.empty(ctx.weight_cache_bytes, dtype=torch.uint8, device=dev)
    B.lsp_layer_prepare_weights(ctx, weights, cache, stream)
    out = dict(weights)
    out["f16_cache"] = cache
    return out


def pad_heads(t: np.ndarray, name: str, n_heads: int, d: int, d_pad: int) -> np.ndarray:
    """Zero-pad every head of a projection tensor from width d to d_pad (lsp_layer_desc.head_dim_logical): rows of
    wq / wk / wv ([heads*d, H]), columns of wo ([H, heads*d]).  Works on weights (uint16 bf16 bits) and gradients."""
    if name == "wo":
        out = np.zeros((t.shape[0], n_heads, d_pad), t.dtype)
        out[:, :, :d] = t.reshape(t.shape[0], n_heads, d)
        return out.reshape(t.shape[0], n_heads * d_pad)
    out = np.zeros((n_heads, d_pad, t.shape[1]), t.dtype)
    out[:, :d, :] = t.reshape(n_heads, d, t.shape[1])
    return out.reshape(n_heads * d_pad, t.shape[1])


def unpad_heads(t: np.ndarray, name: str, n_heads: int, d: int, d_pad: int):
    """Inverse of pad_heads; returns (unpadded tensor, the padding part) so callers can check that the padding is zero."""
    if name == "wo":
        v = t.reshape(t.shape[0], n_heads, d_pad)
        return v[:, :, :d].reshape(t.shape[0], n_heads * d), v[:, :, d:]
    v = t.reshape(n_heads, d_pad, t.shape[1])
    return v[:, :d, :].reshape(n_heads * d, t.shape[1]), v[:, d:, :]


def run_layer(w: synth.Workload, layer: int = 0, grads_init: dict | None = None, weights_bits: dict | None = None, **desc_kw):
    """One lsp_layer_fwd + lsp_layer_bwd on the seeded inputs of workload `w`; returns numpy float32 results.
    grads_init: numpy fp32 arrays the gradient buffers hold before the backward (wgrad_accumulate contexts)."""
    dev = require_cuda()
    ctx = make_ctx(w, **desc_kw)
    buf = LayerBuffers(ctx, w, dev)
    if grads_init is not None:
        for k, v in grads_init.items():
            buf.grads[k].copy_(torch.from_numpy(v))
    weights = upload_weights(weights_bits if weights_bits is not None else synth.layer_weights(w, layer), dev)
    inp = synth.layer_inputs(w)
    x, dy = bf16_to_device(inp["x"], dev), bf16_to_device(inp["dy"], dev)
    B.lsp_layer_fwd(ctx, x, weights, buf.y, buf.saved, buf.ws)
    B.lsp_layer_bwd(ctx, x, dy, weights, buf.saved, buf.dx, buf.grads, buf.ws)
    torch.cuda.synchronize()
    out = dict(y=buf.y.cpu().numpy(), dx=buf.dx.cpu().numpy())
    out.update({"d" + k: v.cpu().numpy() for k, v in buf.grads.items()})
    ctx.close()
    return out


class StackRunner:
    """BASELINE.json config 3: embedding gather, then n_layers x lsp_layer_fwd, then n_layers x lsp_layer_bwd in
    reverse (reading A-11: no final norm / head / loss; the upstream gradient enters at the last layer's output).
    The residual stream between layers is fp32 (in_dtype = LSP_F32); every layer keeps its own `saved` bundle, the
    workspace is shared.  Host-side sequencing only -- every step runs in the library's kernels."""

    def __init__(self, w: synth.Workload, n_layers: int, dev=None, cache_weights: bool = False):
        """cache_weights: hand every layer its fp16 operand cache (lsp_layer_prepare_weights once, here) -- the weights of
        the stack do not change between calls, so no forward launches a weight cast."""
        self.dev = dev or require_cuda()
        self.w, self.L = w, n_layers
        self.ctx = make_ctx(w, in_dtype=B.LSP_F32)
        T, H = w.tokens, w.hidden
        f32 = dict(dtype=torch.float32, device=self.dev)
        self.saved = [torch.empty(self.ctx.saved_bytes, dtype=torch.uint8, device=self.dev) for _ in range(n_layers)]
        self.ws = torch.empty(self.ctx.workspace_bytes, dtype=torch.uint8, device=self.dev)
        self.xs = [torch.empty((T, H), **f32) for _ in range(n_layers + 1)]
        self.d = [torch.empty((T, H), **f32) for _ in range(2)]
        self.weights = [upload_weights(synth.layer_weights(w, layer), self.dev) for layer in range(n_layers)]
        if cache_weights:
            self.weights = [with_weight_cache(self.ctx, wl, self.dev) for wl in self.weights]
        self.grads = {k: torch.empty(s, **f32) for k, s in WEIGHT_SHAPES(w).items()}

    def forward(self, ids: torch.Tensor, table: torch.Tensor, stream=None):
        B.lsp_embed_fwd(self.ctx, ids, table, self.xs[0], stream)
        for l in range(self.L):
            B.lsp_layer_fwd(self.ctx, self.xs[l], self.weights[l], self.xs[l + 1], self.saved[l], self.ws, stream)
        return self.xs[self.L]

    def backward(self, dy32: torch.Tensor, on_layer_grads=None, stream=None):
        """dy32: fp32 [T,H].  on_layer_grads(layer, grads_dict) is called after each layer's backward (the gradient
        buffers are reused by the next layer).  Returns dx0 (gradient w.r.t. the gathered embeddings)."""
        d_in = dy32
        for i, l in enumerate(range(self.L - 1, -1, -1)):
            d_out = self.d[i & 1]
            B.lsp_layer_bwd(self.ctx, self.xs[l], d_in, self.weights[l], self.saved[l], d_out, self.grads, self.ws, stream)
            if on_layer_grads is not None:
                on_layer_grads(l, self.grads)
            d_in = d_out
        return d_in

    def close(self):
        self.ctx.close()
