"""Device-side timing of every BASELINE.json configuration (bench.py covers the headline config 2 only).

    python bench_configs.py [--steps K] [--only cfg2,fwd,packed,cfg3,cfg4,cfg5,table1,table1_30b,adamw,head,gemm]

Prints one JSON line per configuration: ms per fwd+bwd step (CUDA events on the launching stream, after warm-up),
tokens/s and executed TFLOP/s (causal attention FLOPs, SURVEY.md 8(d) convention).  Inputs are the seeded synthetic
tensors of synth.py, resident in HBM.  Every step runs through the C ABI (binding.py); nothing here imports the oracle.
"""
from __future__ import annotations

import argparse
import json
import math

import torch

import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from paper_2510_02483_b200 import binding as B  # noqa: E402
from paper_2510_02483_b200 import harness, synth  # noqa: E402


def _time(fn, steps, warmup=3):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def bench_layer(w, steps, logical_head_dim=0):
    """logical_head_dim: the workload's heads are that wide, zero-padded to w.head_dim (lsp_layer_desc.head_dim_logical);
    the FLOPs returned are the LOGICAL ones (the padding is overhead, not work)."""
    dev = harness.require_cuda()
    ctx = harness.make_ctx(w, head_dim_logical=logical_head_dim)
    buf = harness.LayerBuffers(ctx, w, dev)
    if logical_head_dim:
        wl = w.with_(head_dim=logical_head_dim)
        bits = synth.layer_weights(wl)
        for k, n in dict(wq=w.n_q_heads, wk=w.n_kv_heads, wv=w.n_kv_heads, wo=w.n_q_heads).items():
            bits[k] = harness.pad_heads(bits[k], k, n, logical_head_dim, w.head_dim)
        weights = harness.upload_weights(bits, dev)
    else:
        wl = w
        weights = harness.upload_weights(synth.layer_weights(w), dev)
    weights = harness.with_weight_cache(ctx, weights, dev)          # unchanged between steps: fp16 operand copies made once (as bench.py)
    inp = synth.layer_inputs(w)
    x, dy = harness.bf16_to_device(inp["x"], dev), harness.bf16_to_device(inp["dy"], dev)

    def step():
        B.lsp_layer_fwd(ctx, x, weights, buf.y, buf.saved, buf.ws)
        B.lsp_layer_bwd(ctx, x, dy, weights, buf.saved, buf.dx, buf.grads, buf.ws)
    ms = _time(step, steps)
    ctx.close()
    return ms, synth.layer_flops(wl, causal=True)


def bench_layer_packed(w, steps, cu):
    """cfg-2 layer on packed variable-length sequences (lsp_set_packed_sequences): batch 1, seq = all tokens, sequence
    boundaries `cu`.  FLOPs: GEMMs as usual, causal attention summed over the sequences."""
    dev = harness.require_cuda()
    ctx = harness.make_ctx(w)
    buf = harness.LayerBuffers(ctx, w, dev)
    weights = harness.with_weight_cache(ctx, harness.upload_weights(synth.layer_weights(w), dev), dev)
    inp = synth.layer_inputs(w)
    x, dy = harness.bf16_to_device(inp["x"], dev), harness.bf16_to_device(inp["dy"], dev)
    B.lsp_set_packed_sequences(ctx, cu)

    def step():
        B.lsp_layer_fwd(ctx, x, weights, buf.y, buf.saved, buf.ws)
        B.lsp_layer_bwd(ctx, x, dy, weights, buf.saved, buf.dx, buf.grads, buf.ws)
    ms = _time(step, steps)
    ctx.close()
    one = w.with_(seq=1)
    gemm = synth.layer_flops(one, causal=True) - 3.5 * synth.attn_flops_fwd(one, causal=True)
    attn = sum(3.5 * synth.attn_flops_fwd(w.with_(batch=1, seq=b - a), causal=True) for a, b in zip(cu, cu[1:]))
    return ms, gemm * w.tokens + attn


def bench_layer_fwd_only(w, steps, infer=False):
    """Forward pass alone (the forward-only variant, prefill-style), device-resident: lsp_layer_fwd, or
    lsp_layer_fwd_infer (nothing kept for a backward pass)."""
    dev = harness.require_cuda()
    ctx = harness.make_ctx(w)
    buf = harness.LayerBuffers(ctx, w, dev)
    weights = harness.with_weight_cache(ctx, harness.upload_weights(synth.layer_weights(w), dev), dev)
    x = harness.bf16_to_device(synth.layer_inputs(w)["x"], dev)
    fn = B.lsp_layer_fwd_infer if infer else B.lsp_layer_fwd
    ms = _time(lambda: fn(ctx, x, weights, buf.y, buf.saved, buf.ws), steps)
    ctx.close()
    return ms, synth.layer_flops(w, causal=True) / 3.0 - synth.attn_flops_fwd(w, causal=True) * (3.5 / 3.0 - 1.0)


def bench_stack(w, steps):
    """Config 3: embedding gather + n_layers x (fwd) + n_layers x (bwd); every layer has its own seeded weights."""
    dev = harness.require_cuda()
    run = harness.StackRunner(w, w.n_layers, dev, cache_weights=True)
    s = synth.stack_inputs(w)
    ids = torch.from_numpy(s["ids"]).to(dev)
    table = harness.bf16_to_device(s["embedding"], dev)
    dy = harness.bf16_to_device(synth.layer_inputs(w)["dy"], dev).float()

    def step():
        run.forward(ids, table)
        run.backward(dy)
    ms = _time(step, steps, warmup=2)
    run.close()
    return ms, w.n_layers * synth.layer_flops(w, causal=True)


def bench_sdpa(w, steps):
    dev = harness.require_cuda()
    ctx = harness.make_ctx(w, use_rope=False)
    t = {k: harness.bf16_to_device(v, dev) for k, v in synth.attn_inputs(w).items()}
    Bz, S, nq, nkv, d = w.batch, w.seq, w.n_q_heads, w.n_kv_heads, w.head_dim
    o = torch.empty((Bz, S, nq, d), dtype=torch.float32, device=dev)
    lse = torch.empty((Bz, nq, S), dtype=torch.float32, device=dev)
    dq = torch.empty_like(o)
    dk = torch.empty((Bz, S, nkv, d), dtype=torch.float32, device=dev)
    dv = torch.empty_like(dk)
    ws = torch.empty(ctx.workspace_bytes, dtype=torch.uint8, device=dev)

    def step():
        B.lsp_sdpa_fwd(ctx, t["q"], t["k"], t["v"], o, lse, ws)
        B.lsp_sdpa_bwd(ctx, t["q"], t["k"], t["v"], o, lse, t["dO"], dq, dk, dv, ws)
    ms = _time(step, steps)
    ctx.close()
    fwd = 4.0 * d * nq * Bz * S * (S + 1) / 2.0
    return ms, 3.5 * fwd


def bench_adamw(w, steps):
    """Optimizer step (lsp_adamw_step) on the nine tensors of one layer of workload `w`: HBM-bound, 34 algorithmic bytes
    per parameter (norm pass 4 B; update reads g, p, m, v 16 B, writes p, m, v and the bf16 weight 14 B)."""
    dev = harness.require_cuda()
    ctx = harness.make_ctx(synth.CFG1_TINY)
    tensors = []
    for k, shape in harness.WEIGHT_SHAPES(w).items():
        f = lambda: torch.randn(shape, dtype=torch.float32, device=dev) * 0.02
        tensors.append(dict(grad=f(), master=f(), m=torch.zeros(shape, dtype=torch.float32, device=dev),
                            v=torch.zeros(shape, dtype=torch.float32, device=dev),
                            weight=torch.empty(shape, dtype=torch.bfloat16, device=dev), decay=len(shape) == 2))
    gn = torch.zeros(2, dtype=torch.float32, device=dev)
    state = {"t": 0}

    def step():
        state["t"] += 1
        B.lsp_adamw_step(ctx, tensors, lr=B.lsp_lr_cosine(state["t"]), step=state["t"], gnorm_out=gn)
    ms = _time(step, steps)
    ctx.close()
    nparam = sum(t["master"].numel() for t in tensors)
    return ms, nparam


def bench_head(w, steps):
    """Model head of config 3 (lsp_head_fwd_bwd: final RMSNorm + LM head [T,H] x [H,V] + cross-entropy, fwd and bwd) and
    the embedding backward (lsp_embed_bwd), T = batch * seq tokens, V = the workload's vocabulary."""
    dev = harness.require_cuda()
    ctx = harness.make_ctx(w, in_dtype=B.LSP_F32)
    T, H, V = w.tokens, w.hidden, w.vocab
    s = synth.stack_inputs(w)
    ids = torch.from_numpy(s["ids"]).to(dev)
    x = torch.randn((T, H), dtype=torch.float32, device=dev)
    g = torch.ones(H, dtype=torch.bfloat16, device=dev)
    wh = harness.bf16_to_device(s["embedding"], dev)            # an untied head of the embedding's shape and distribution
    loss = torch.zeros(1, dtype=torch.float32, device=dev); lse = torch.empty(T, dtype=torch.float32, device=dev)
    dx = torch.empty((T, H), dtype=torch.float32, device=dev); dg = torch.empty(H, dtype=torch.float32, device=dev)
    dw = torch.empty((V, H), dtype=torch.float32, device=dev)
    ws = torch.empty(B.lsp_head_workspace_bytes(ctx, V), dtype=torch.uint8, device=dev)
    ms_head = _time(lambda: B.lsp_head_fwd_bwd(ctx, x, g, wh, ids, V, loss, lse, dx, dg, dw, ws), steps)
    ms_emb = _time(lambda: B.lsp_embed_bwd(ctx, ids, dx, V, dw), steps)
    out = dict(ms_head=ms_head, ms_embed_bwd=ms_emb, loss=float(loss.cpu()), flops=3 * 2.0 * T * V * H)
    ctx.close()
    return out


def gemm_shapes(w):
    """The 12 GEMMs of one layer step of workload `w` as (stage, lsp_gemm op, M, N, K)."""
    T, H, F = w.tokens, w.hidden, w.ffn
    Nq, Nqkv = w.n_q_heads * w.head_dim, (w.n_q_heads + 2 * w.n_kv_heads) * w.head_dim
    return [("gemm_qkv", 0, T, Nqkv, H), ("gemm_oproj", 0, T, H, Nq), ("gemm_gateup", 0, T, 2 * F, H), ("gemm_down", 0, T, H, F),
            ("wgrad_down", 2, H, F, T), ("dgrad_down", 1, T, F, H), ("wgrad_gateup", 2, 2 * F, H, T), ("dgrad_gateup", 1, T, H, 2 * F),
            ("wgrad_oproj", 2, H, Nq, T), ("dgrad_oproj", 1, T, Nq, H), ("wgrad_qkv", 2, Nqkv, H, T), ("dgrad_qkv", 1, T, H, Nqkv)]


def bench_gemm_shapes(w, steps):
    """Every GEMM shape of the layer step, alone: lsp_gemm (the tcgen05 kernel with its plain fp32-store epilogue; fp16 operands
    as in the layer, and bf16 operands) against cuBLAS through torch (bf16 in / bf16 out, fp16 in / fp16 out, and bf16 in / fp32
    out where this torch offers out_dtype) on the same N(0,1) data, timed back to back in turns on the same GPU in the same
    power state (under the pool's power cap the operand FORMAT matters: the clock settles where the board draws its cap).  cuBLAS is the library yardstick of the
    roofline (MEASURED_PEAKS.json times it at 8192^3 only); the in-step GEMMs carry fused epilogues on top of this."""
    dev = harness.require_cuda()
    ctx = harness.make_ctx(synth.CFG1_TINY)
    rows = []
    for name, op, M, N, K in gemm_shapes(w):
        a_shape = (K, M) if op == 2 else (M, K)
        b_shape = (N, K) if op == 0 else (K, N)
        a16 = torch.randn(a_shape, dtype=torch.float32, device=dev).to(torch.float16)
        b16 = torch.randn(b_shape, dtype=torch.float32, device=dev).to(torch.float16)
        ab, bb = a16.to(torch.bfloat16), b16.to(torch.bfloat16)
        c32 = torch.empty((M, N), dtype=torch.float32, device=dev)
        cb = torch.empty((M, N), dtype=torch.bfloat16, device=dev)
        ta = ab.t() if op == 2 else ab
        tb = bb.t() if op == 0 else bb

        th = a16.t() if op == 2 else a16
        tbh = b16.t() if op == 0 else b16
        ch = torch.empty((M, N), dtype=torch.float16, device=dev)

        def ours():
            B.lsp_gemm(ctx, op, M, N, K, a16, a_shape[1], B.LSP_F16, b16, b_shape[1], B.LSP_F16, c32, N)

        def ours_bf16():
            B.lsp_gemm(ctx, op, M, N, K, ab, a_shape[1], B.LSP_BF16, bb, b_shape[1], B.LSP_BF16, c32, N)

        def cublas_bf16():
            torch.mm(ta, tb, out=cb)

        def cublas_f16():
            torch.mm(th, tbh, out=ch)

        def cublas_f32():
            torch.mm(ta, tb, out_dtype=torch.float32, out=c32)
        try:
            cublas_f32()
            have_f32 = True
        except (TypeError, RuntimeError):
            have_f32 = False
        fns = {"ours": ours, "ours_bf16_operands": ours_bf16, "cublas_bf16_out": cublas_bf16, "cublas_f16_in_out": cublas_f16}
        if have_f32:
            fns["cublas_f32_out"] = cublas_f32
        best = {k: 1e9 for k in fns}
        for _ in range(3):                                   # in turns: the same thermal / power state for all
            for k, f in fns.items():
                best[k] = min(best[k], _time(f, steps))
        fl = 2.0 * M * N * K
        row = {"config": "gemm_" + w.name, "stage": name, "op": op, "M": M, "N": N, "K": K}
        for k, v in best.items():
            row[k + "_ms"] = round(v, 4)
            row[k + "_tflops"] = round(fl / v / 1e9, 1)
        rows.append(row)
        print(json.dumps(row), flush=True)
        del a16, b16, ab, bb, c32, cb, ch
        torch.cuda.empty_cache()
    keys = [k for k in rows[0] if k.endswith("_ms")]
    print(json.dumps({"config": "gemm_" + w.name, "stage": "sum of the 12", **{k: round(sum(r[k] for r in rows), 4) for k in keys}}), flush=True)
    ctx.close()


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--only", default="cfg2,fwd,packed,cfg3,cfg4,cfg5,table1,table1_30b,adamw,head,gemm")
    args = ap.parse_args(argv)
    B.lib()
    only = set(args.only.split(","))
    jobs = []
    if "cfg2" in only:
        jobs.append((synth.CFG2_3B_LAYER, bench_layer))
    if "packed" in only:      # 16384 tokens of the 3B-shape layer as ONE row holding 7 sequences of 333 ... 6000 tokens
        cu = [0, 333, 1500, 5596, 6000, 12000, 14048, 16384]
        wp = synth.CFG2_3B_LAYER.with_(name="cfg2_3b_layer_packed_7_sequences", batch=1, seq=16384)
        jobs.append((wp, lambda w, steps: bench_layer_packed(w, steps, cu)))
        jobs.append((wp.with_(name="cfg2_3b_layer_one_sequence_of_16384"), lambda w, steps: bench_layer_packed(w, steps, [0, 16384])))
    if "fwd" in only:
        jobs.append((synth.CFG2_3B_LAYER.with_(name="cfg2_3b_layer_forward_only"), bench_layer_fwd_only))
        jobs.append((synth.CFG2_3B_LAYER.with_(name="cfg2_3b_layer_forward_infer"), lambda w, steps: bench_layer_fwd_only(w, steps, True)))
    if "cfg4" in only:
        jobs.append((synth.CFG4_30B_LAYER, bench_layer))
    if "table1" in only:      # the paper's own Table-1 3B layer shape: hidden 2048, 16q / 2kv, FFN 11008
        jobs.append((synth.Workload("table1_3b_layer", 6, 4, 4096, 2048, 16, 2, 128, 11008, 1e-5, 10000.0), bench_layer))
    if "table1_30b" in only:  # Table-1 30B layer as printed: hidden 6656, 64 MHA heads of width 104 (zero-padded to 128), FFN 17920
        w30 = synth.Workload("table1_30b_layer_64x104_padded", 7, 2, 4096, 6656, 64, 64, 128, 17920, 1e-5, 10000.0)
        jobs.append((w30, lambda w, steps: bench_layer(w, steps, logical_head_dim=104)))
    if "cfg3" in only:
        jobs.append((synth.CFG3_3B_STACK, bench_stack))
    if "cfg5" in only:
        jobs += [(w, bench_sdpa) for w in synth.CFG5_ATTN]
    if "adamw" in only:
        for w in (synth.CFG2_3B_LAYER, synth.CFG4_30B_LAYER):
            ms, nparam = bench_adamw(w, args.steps)
            print(json.dumps({"config": "adamw_" + w.name, "params": nparam, "ms_per_step": round(ms, 4),
                              "algorithmic_GB_per_s": round(34.0 * nparam / (ms * 1e-3) / 1e9, 1)}), flush=True)
            torch.cuda.empty_cache()
    if "gemm" in only:
        bench_gemm_shapes(synth.CFG2_3B_LAYER, max(args.steps, 20))
    if "head" in only:
        w = synth.CFG3_3B_STACK
        r = bench_head(w, min(args.steps, 5))
        print(json.dumps({"config": "head_" + w.name, "tokens": w.tokens, "vocab": w.vocab, "ms_head_fwd_bwd": round(r["ms_head"], 4),
                          "gemm_tflops": round(r["flops"] / (r["ms_head"] * 1e-3) / 1e12, 1), "loss": round(r["loss"], 4),
                          "ln_vocab": round(math.log(w.vocab), 4), "ms_embed_bwd": round(r["ms_embed_bwd"], 4)}), flush=True)
        torch.cuda.empty_cache()
    for w, fn in jobs:
        ms, flops = fn(w, max(2, args.steps if fn is not bench_stack else min(args.steps, 3)))
        print(json.dumps({"config": w.name, "batch": w.batch, "seq": w.seq, "tokens": w.tokens, "ms_per_step": round(ms, 4),
                          "tokens_per_s": round(w.tokens / (ms * 1e-3), 1), "tflops_executed": round(flops / (ms * 1e-3) / 1e12, 1)}),
              flush=True)
        torch.cuda.empty_cache()
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
