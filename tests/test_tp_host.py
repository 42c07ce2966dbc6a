"""Host logic of paper_2510_02483_b200/tp.py on CPU: slicing by heads / FFN columns, re-assembly of gradients, and the
algebra the tensor-parallel layer rests on -- with the fp64 oracle standing in for the kernels: the attention and MLP
blocks of the sliced layers, with the residual counted once, add up to the blocks of the whole layer."""
import numpy as np
import pytest

from oracle import lspref as R
from paper_2510_02483_b200 import synth, tp as TP

W = synth.Workload("tp_cpu", 58, 2, 12, 32, 4, 2, 8, 48, 1e-5, 10000.0)


def _weights(rng):
    H, d = W.hidden, W.head_dim
    sh = dict(wq=(W.n_q_heads * d, H), wk=(W.n_kv_heads * d, H), wv=(W.n_kv_heads * d, H), wo=(H, W.n_q_heads * d),
              w_gate=(W.ffn, H), w_up=(W.ffn, H), w_down=(H, W.ffn), g_attn=(H,), g_mlp=(H,))
    return {k: (1.0 + 0.1 * rng.standard_normal(s)) if k.startswith("g_") else 0.3 * rng.standard_normal(s) for k, s in sh.items()}


def test_shard_and_unshard_round_trip():
    rng = np.random.default_rng(1)
    full = _weights(rng)
    for tp in (1, 2):
        parts = [TP.shard_tensors(full, W, tp, r) for r in range(tp)]
        back = TP.unshard_grads(parts, W)
        for k in full:
            if k.startswith("g_"):
                np.testing.assert_allclose(back[k], tp * full[k])           # gain gradients are SUMMED over ranks
            else:
                np.testing.assert_array_equal(back[k], full[k])
    sw = TP.shard_workload(W.with_(ffn=64), 2)
    assert (sw.n_q_heads, sw.n_kv_heads, sw.ffn) == (2, 1, 32)
    with pytest.raises(ValueError):
        TP.shard_workload(W, 3)


def test_sliced_blocks_add_up_to_the_layer():
    rng = np.random.default_rng(2)
    full = _weights(rng)
    x = rng.standard_normal((W.tokens, W.hidden)); dy = rng.standard_normal((W.tokens, W.hidden))
    cfg = R.LayerShape(W.batch, W.seq, W.hidden, W.n_q_heads, W.n_kv_heads, W.head_dim, W.ffn, W.rms_eps, W.rope_base, 0, True)
    ref = R.layer_fwd_bwd(x, dy, full, cfg)
    tp = 2
    sw = TP.shard_workload(W, tp)
    scfg = R.LayerShape(sw.batch, sw.seq, sw.hidden, sw.n_q_heads, sw.n_kv_heads, sw.head_dim, sw.ffn, sw.rms_eps, sw.rope_base, 0, True)
    parts = [TP.shard_tensors(full, W, tp, r) for r in range(tp)]
    # every rank computes residual + partial; the residual is counted once (residual_scale 1 on rank 0 only)
    a_r, c_a = zip(*[R.attn_block_fwd(x, p, scfg) for p in parts])
    a = sum(a_r) - (tp - 1) * x
    np.testing.assert_allclose(a, ref["a"], rtol=1e-11, atol=1e-12)
    y_r, c_m = zip(*[R.mlp_block_fwd(a, p, scfg) for p in parts])
    y = sum(y_r) - (tp - 1) * a
    np.testing.assert_allclose(y, ref["y"], rtol=1e-11, atol=1e-12)
    da_r, g_m = zip(*[R.mlp_block_bwd(dy, p, scfg, c) for p, c in zip(parts, c_m)])
    da = sum(da_r) - (tp - 1) * dy
    np.testing.assert_allclose(da, ref["da"], rtol=1e-10, atol=1e-12)
    dx_r, g_a = zip(*[R.attn_block_bwd(da, p, scfg, c) for p, c in zip(parts, c_a)])
    dx = sum(dx_r) - (tp - 1) * da
    np.testing.assert_allclose(dx, ref["dx"], rtol=1e-10, atol=1e-12)
    grads = TP.unshard_grads([dict(ga, **gm) for ga, gm in zip(g_a, g_m)], W)
    for k, v in grads.items():
        np.testing.assert_allclose(v, ref["d" + k], rtol=1e-9, atol=1e-12, err_msg=k)
