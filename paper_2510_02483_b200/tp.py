"""Tensor parallelism of one decoder layer: every rank holds a slice of the heads
(rows of Wq / Wk / Wv, columns of Wo) and of the FFN columns (rows of W_gate / W_up, columns of W_down) and runs the
SAME library kernels on its slice -- a layer with n_q_heads / tp, n_kv_heads / tp, ffn / tp.  Each block then yields a
PARTIAL sum over the sliced contraction, and the four exchange steps of the layer are all-reduces of a [T, H] fp32 tensor:

    forward   a = sum_r a_r   (after the O-projection),   y = sum_r y_r   (after the down-projection)
    backward  da = sum_r da_r (after the gate/up dgrads), dx = sum_r dx_r (after the QKV dgrad)

The residual branches must enter the sum once: rank 0 runs with residual_scale 1, the others with 0 (lsp_layer_desc), so
no correction pass exists.  RMSNorm is recomputed on every rank from the full input; its backward is linear in the
partial gradient, so the partial dx's add up, and the gain gradients are all-reduced with the other [H] vectors.
Weight gradients stay local (each rank owns its slice).

One process per GPU with torch.distributed (NCCL over NVLink 5 / NVSwitch); without a process group the all-reduces are
the identity, and `phases()` lets a test drive several shards one after the other on one GPU and add their partials.

UNMEASURED ON HARDWARE: rounds 1 and 2 had one GPU; the shards' algebra is tested (sequentially, on one GPU), the four
all-reduces have never run over NCCL and nothing is claimed about their cost.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

from . import binding as B
from . import harness, synth

_ROWS = dict(wq="q", wk="kv", wv="kv", w_gate="f", w_up="f")      # sliced along rows ([out, in]: output features)
_COLS = dict(wo="q", w_down="f")                                  # sliced along columns (input features)


def shard_workload(w: synth.Workload, tp: int) -> synth.Workload:
    if w.n_q_heads % tp or w.n_kv_heads % tp or w.ffn % (8 * tp):
        raise ValueError("heads and ffn / 8 must divide by the tensor-parallel degree")
    return w.with_(n_q_heads=w.n_q_heads // tp, n_kv_heads=w.n_kv_heads // tp, ffn=w.ffn // tp)


def _span(kind: str, w: synth.Workload, tp: int, r: int):
    n = dict(q=w.n_q_heads * w.head_dim, kv=w.n_kv_heads * w.head_dim, f=w.ffn)[kind] // tp
    return slice(r * n, (r + 1) * n)


def shard_tensors(full: dict, w: synth.Workload, tp: int, r: int) -> dict:
    """Slice of rank r of the nine tensors of a layer (numpy arrays of any dtype: weights as bf16 bits, or gradients)."""
    out = {}
    for k, v in full.items():
        if k in _ROWS:
            out[k] = np.ascontiguousarray(v[_span(_ROWS[k], w, tp, r), :])
        elif k in _COLS:
            out[k] = np.ascontiguousarray(v[:, _span(_COLS[k], w, tp, r)])
        else:
            out[k] = v
    return out


def unshard_grads(parts: list, w: synth.Workload) -> dict:
    """Full-layer gradients from the per-rank ones: slices concatenated, gain gradients summed."""
    out = {}
    for k in parts[0]:
        if k in _ROWS:
            out[k] = np.concatenate([p[k] for p in parts], axis=0)
        elif k in _COLS:
            out[k] = np.concatenate([p[k] for p in parts], axis=1)
        else:
            out[k] = sum(p[k] for p in parts)
    return out


def all_reduce_(t: torch.Tensor, group=None) -> torch.Tensor:
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


class TPLayer:
    """Rank `rank` of `tp` of one layer of workload `w` (the FULL layer shape).  x / dy / every exchanged tensor: fp32 [T, H]."""

    def __init__(self, w: synth.Workload, tp: int, rank: int, weights_bits: dict, dev=None, group=None):
        self.dev = dev or harness.require_cuda()
        self.w, self.tp, self.rank, self.group = w, tp, rank, group
        self.ws_ = shard_workload(w, tp)
        self.ctx = harness.make_ctx(self.ws_, in_dtype=B.LSP_F32, residual_scale=1.0 if rank == 0 else 0.0)
        self.buf = harness.LayerBuffers(self.ctx, self.ws_, self.dev)
        self.weights = harness.upload_weights(shard_tensors(weights_bits, w, tp, rank), self.dev)
        T, H = w.tokens, w.hidden
        self.a = torch.empty((T, H), dtype=torch.float32, device=self.dev)
        self.da = torch.empty((T, H), dtype=torch.float32, device=self.dev)

    # the four phases; each returns this rank's PARTIAL [T, H] result (to be summed over ranks)
    def attn_fwd(self, x):
        B.lsp_attn_fwd(self.ctx, x, self.weights, self.a, self.buf.saved, self.buf.ws)
        return self.a

    def mlp_fwd(self, a):
        B.lsp_mlp_fwd(self.ctx, a, self.weights, self.buf.y, self.buf.saved, self.buf.ws)
        return self.buf.y

    def mlp_bwd(self, a, dy):
        B.lsp_mlp_bwd(self.ctx, a, dy, self.weights, self.buf.saved, self.da, self.buf.grads, self.buf.ws)
        return self.da

    def attn_bwd(self, x, da):
        B.lsp_attn_bwd(self.ctx, x, da, self.weights, self.buf.saved, self.buf.dx, self.buf.grads, self.buf.ws)
        return self.buf.dx

    def step(self, x, dy):
        """Forward + backward of the layer on this rank with the four all-reduces; returns (y, dx), full on every rank.
        Gain gradients are all-reduced too; the weight-gradient slices stay in self.buf.grads."""
        a = all_reduce_(self.attn_fwd(x), self.group)
        y = all_reduce_(self.mlp_fwd(a), self.group)
        da = all_reduce_(self.mlp_bwd(a, dy), self.group)
        dx = all_reduce_(self.attn_bwd(x, da), self.group)
        all_reduce_(self.buf.grads["g_attn"], self.group)
        all_reduce_(self.buf.grads["g_mlp"], self.group)
        return y, dx

    def close(self):
        self.ctx.close()


def phases(shards: list, x: torch.Tensor, dy: torch.Tensor):
    """Drive all shards of a layer one after the other on ONE device (tests): after each phase the partial results are
    added in rank order, which is what the all-reduce of `TPLayer.step` computes across devices.  Returns (y, dx)."""
    def total(parts):
        s = parts[0].clone()
        for p in parts[1:]:
            s += p
        return s
    a = total([s.attn_fwd(x) for s in shards])
    y = total([s.mlp_fwd(a) for s in shards])
    da = total([s.mlp_bwd(a, dy) for s in shards])
    dx = total([s.attn_bwd(x, da) for s in shards])
    return y, dx
