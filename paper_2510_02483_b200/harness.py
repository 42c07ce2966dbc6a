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


def make_ctx(w: synth.Workload, use_rope=True, in_dtype=B.LSP_BF16) -> B.Ctx:
    return B.Ctx(batch=w.batch, seq=w.seq, hidden=w.hidden, n_q_heads=w.n_q_heads, n_kv_heads=w.n_kv_heads,
                 head_dim=w.head_dim, ffn=w.ffn, rms_eps=w.rms_eps, rope_base=w.rope_base, use_rope=use_rope,
                 in_dtype=in_dtype, device=torch.cuda.current_device())


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


def run_layer(w: synth.Workload, layer: int = 0):
    """One lsp_layer_fwd + lsp_layer_bwd on the seeded inputs of workload `w`; returns numpy float32 results."""
    dev = require_cuda()
    ctx = make_ctx(w)
    buf = LayerBuffers(ctx, w, dev)
    weights = upload_weights(synth.layer_weights(w, layer), dev)
    inp = synth.layer_inputs(w)
    x, dy = bf16_to_device(inp["x"], dev), bf16_to_device(inp["dy"], dev)
    B.lsp_layer_fwd(ctx, x, weights, buf.y, buf.saved, buf.ws)
    B.lsp_layer_bwd(ctx, x, dy, weights, buf.saved, buf.dx, buf.grads, buf.ws)
    torch.cuda.synchronize()
    out = dict(y=buf.y.cpu().numpy(), dx=buf.dx.cpu().numpy())
    out.update({"d" + k: v.cpu().numpy() for k, v in buf.grads.items()})
    ctx.close()
    return out
