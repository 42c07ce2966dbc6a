"""Seeded synthetic inputs for the decoder-layer workloads (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path's callers (tests, bench.py) and the oracle's callers, and
therefore holds none of the method's arithmetic: only shapes, seeds, a normal sampler and the
bf16 storage rounding of the *inputs*.  Recipe (fixed before any result existed):

  rng = numpy.random.default_rng(SeedSequence([2510, 2483, cfg, layer, tensor_id]))
  value = bf16_rne(rng.standard_normal(float32) * scale [+ 1 for gains])

The paper trained on SlimPajama-627B with a 32k SentencePiece vocabulary; neither is
needed: a dense layer's arithmetic and throughput do not depend on token content, so seeded N(0,1)
activations / N(0,0.02) weights of the workload's shapes stand in (BASELINE.json configs).
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

TENSOR_ID = dict(x=0, dy=1, wq=2, wk=3, wv=4, wo=5, w_gate=6, w_up=7, w_down=8, g_attn=9, g_mlp=10,
                 ids=11, embedding=12, q=13, k=14, v=15, dO=16, w_head=17, g_final=18)
WEIGHT_NAMES = ("wq", "wk", "wv", "wo", "g_attn", "w_gate", "w_up", "w_down", "g_mlp")


@dataclass(frozen=True)
class Workload:
    name: str
    cfg_id: int
    batch: int
    seq: int
    hidden: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    ffn: int
    rms_eps: float = 1e-5
    rope_base: float = 10000.0
    n_layers: int = 1
    vocab: int = 0

    @property
    def tokens(self):
        return self.batch * self.seq

    def with_(self, **kw):
        return replace(self, **kw)


# BASELINE.json `configs` (index = position in that list; cfg_id = index + 1 as in SURVEY 8(d)).
CFG1_TINY = Workload("cfg1_tiny", 1, 1, 128, 256, 4, 2, 64, 688, 1e-5, 10000.0)
CFG2_3B_LAYER = Workload("cfg2_3b_layer", 2, 4, 4096, 3072, 24, 8, 128, 8192, 1e-5, 500000.0)
CFG3_3B_STACK = Workload("cfg3_3b_stack", 3, 2, 4096, 3072, 24, 8, 128, 8192, 1e-5, 500000.0, 28, 128256)
CFG4_30B_LAYER = Workload("cfg4_30b_layer", 4, 2, 4096, 6656, 52, 52, 128, 17920, 1e-5, 10000.0)
CFG5_ATTN = tuple(Workload(f"cfg5_attn_s{s}", 5, 32768 // s, s, 3072, 24, 8, 128, 8192) for s in (1024, 4096, 8192, 16384))


def layer_flops(w: Workload, causal: bool = True) -> float:
    """Executed FLOPs of one layer fwd+bwd (GEMM bwd = 2x fwd, attention bwd = 2.5x fwd)."""
    T, H, F = w.tokens, w.hidden, w.ffn
    nqd, nkvd = w.n_q_heads * w.head_dim, w.n_kv_heads * w.head_dim
    gemm_fwd = 2.0 * T * (H * (nqd + 2 * nkvd) + nqd * H + 3 * H * F)
    attn_fwd = attn_flops_fwd(w, causal)
    return 3.0 * gemm_fwd + 3.5 * attn_fwd


def attn_flops_fwd(w: Workload, causal: bool = True) -> float:
    full = 4.0 * w.batch * w.n_q_heads * w.seq * w.seq * w.head_dim
    return full * (w.seq + 1) / (2.0 * w.seq) if causal else full


# ----------------------------------------------------------------------------- bf16 storage helpers
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 -> bfloat16 bit pattern (uint16), round-to-nearest-even. Inputs are finite."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounded = u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))
    return (rounded >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return bf16_bits_to_f32(b).astype(np.float64)


def _rng(cfg_id: int, layer: int, name: str):
    return np.random.default_rng(np.random.SeedSequence([2510, 2483, cfg_id, layer, TENSOR_ID[name]]))


def normal_bf16(cfg_id: int, layer: int, name: str, shape, scale: float, offset: float = 0.0) -> np.ndarray:
    """bf16 bit patterns (uint16) of offset + scale*N(0,1), seeded by (cfg, layer, tensor name)."""
    v = _rng(cfg_id, layer, name).standard_normal(size=shape, dtype=np.float32) * np.float32(scale)
    if offset:
        v = v + np.float32(offset)
    return f32_to_bf16_bits(v)


def layer_weights(w: Workload, layer: int = 0) -> dict:
    """The nine parameter tensors of one layer as bf16 bit patterns, [out,in] row-major.

    Projection weights 0.02*N(0,1); gains 1 + 0.1*N(0,1) (reading A-10).
    """
    H, F = w.hidden, w.ffn
    nqd, nkvd = w.n_q_heads * w.head_dim, w.n_kv_heads * w.head_dim
    shapes = dict(wq=(nqd, H), wk=(nkvd, H), wv=(nkvd, H), wo=(H, nqd), w_gate=(F, H), w_up=(F, H), w_down=(H, F))
    out = {k: normal_bf16(w.cfg_id, layer, k, s, 0.02) for k, s in shapes.items()}
    out["g_attn"] = normal_bf16(w.cfg_id, layer, "g_attn", (H,), 0.1, 1.0)
    out["g_mlp"] = normal_bf16(w.cfg_id, layer, "g_mlp", (H,), 0.1, 1.0)
    return out


def layer_inputs(w: Workload) -> dict:
    """x and upstream gradient dy, [T,H] bf16 bit patterns ~ N(0,1)."""
    return dict(x=normal_bf16(w.cfg_id, 0, "x", (w.tokens, w.hidden), 1.0),
                dy=normal_bf16(w.cfg_id, 0, "dy", (w.tokens, w.hidden), 1.0))


def attn_inputs(w: Workload) -> dict:
    """Q,K,V,dO ~ N(0,1) bf16 for the attention-only sweep (cfg 5); `layer` slot carries seq so each S differs."""
    B, S, d = w.batch, w.seq, w.head_dim
    mk = lambda n, h: normal_bf16(w.cfg_id, S, n, (B, S, h, d), 1.0)
    return dict(q=mk("q", w.n_q_heads), k=mk("k", w.n_kv_heads), v=mk("v", w.n_kv_heads), dO=mk("dO", w.n_q_heads))


def stack_inputs(w: Workload) -> dict:
    """Token ids uniform over the vocab, bf16 embedding table 0.02*N(0,1), upstream dy ~ N(0,1) (cfg 3)."""
    ids = _rng(w.cfg_id, 0, "ids").integers(0, w.vocab, size=(w.tokens,), dtype=np.int32)
    return dict(ids=ids,
                embedding=normal_bf16(w.cfg_id, 0, "embedding", (w.vocab, w.hidden), 0.02),
                dy=normal_bf16(w.cfg_id, 0, "dy", (w.tokens, w.hidden), 1.0))
