"""One pre-training iteration of a Llama model on one B200, sequenced over the C ABI:

    embedding gather -> n_layers x lsp_layer_fwd -> lsp_head_fwd_bwd (final RMSNorm, LM head, cross-entropy, gradients)
    -> n_layers x lsp_layer_bwd -> lsp_embed_bwd -> lsp_adamw_step over every tensor of the model (one global norm).

Host-side sequencing and buffer ownership only: every step runs in the library's kernels, on one stream, with no host
synchronisation inside an iteration (the loss stays on the device until the caller reads it).  Weights are bf16 for the
kernels with fp32 master copies and moments for the optimizer (Table 2).

    python -m paper_2510_02483_b200.pretrain [--layers L] [--steps K]     # timing of the config-3 model, synthetic batch
"""
from __future__ import annotations

import argparse
import json

import torch

from . import binding as B
from . import dp, harness, replicas, synth


class PretrainStep:
    def __init__(self, w: synth.Workload, n_layers: int, vocab: int, dev=None, weights=None, embedding=None, head=None, g_final=None,
                 world: int = 1, group=None, micro_batches: int = 1, recompute: bool = False,
                 zero1: bool = False, rank: int = 0):
        """weights: optional list of per-layer dicts of bf16 bit patterns (synth.layer_weights layout); embedding / head:
        bf16 bit patterns [vocab, H]; g_final: bf16 bits [H].  Defaults: the seeded synthetic tensors of synth.py.
        `w` is one MICRO-batch of this rank's shard; micro_batches > 1: gradient accumulation (the paper's global batch of
        256 sequences, Table 2, does not fit one step) -- the first micro-batch overwrites the gradient buffers,
        the others run on a second context created with wgrad_accumulate = 1; world > 1: data-parallel replicas (dp.py);
        recompute: keep only every layer's INPUT from the forward pass and re-run the layer's forward in front of its
        backward (one shared `saved` buffer instead of n_layers: activation memory / n_layers for one more forward);
        zero1: optimizer state sharded over the `world` replicas (dp.Zero1State), `rank` = this replica."""
        self.dev = dev or harness.require_cuda()
        if world > 1:
            # The persistent GEMMs cut the last wave's tiles into K-slices whose consumer CTA pairs wait for producer pairs of
            # the SAME grid: safe while the whole grid is co-resident, which nothing guarantees once a collective's kernels
            # hold SMs at the same time (never run on more than one GPU: DESIGN.md section 14).  Data-parallel only until then.
            import os
            os.environ.setdefault("LSP_GEMM_STREAMK", "0")
        self.w, self.L, self.V = w, n_layers, vocab
        self.ctx = harness.make_ctx(w, in_dtype=B.LSP_F32)
        self.n_micro = micro_batches
        self.ctx_acc = harness.make_ctx(w, in_dtype=B.LSP_F32, wgrad_accumulate=True) if micro_batches > 1 else None
        T, H = w.tokens, w.hidden
        f32 = dict(dtype=torch.float32, device=self.dev)
        self.recompute = recompute
        shared = torch.empty(self.ctx.saved_bytes, dtype=torch.uint8, device=self.dev) if recompute else None
        self.saved = [shared if recompute else torch.empty(self.ctx.saved_bytes, dtype=torch.uint8, device=self.dev)
                      for _ in range(n_layers)]
        self.ws = torch.empty(max(self.ctx.workspace_bytes, B.lsp_head_workspace_bytes(self.ctx, vocab)), dtype=torch.uint8, device=self.dev)
        self.xs = [torch.empty((T, H), **f32) for _ in range(n_layers + 1)]
        self.d = [torch.empty((T, H), **f32) for _ in range(2)]
        self._loss_buf = torch.zeros((micro_batches, 4), **f32)      # one 16-byte aligned slot per micro-batch
        self.micro_losses = self._loss_buf[:, 0]
        self.loss = self._loss_buf[0, 0:1]
        self.lse = torch.empty(T, **f32)
        self.gnorm = torch.zeros(2, **f32)
        # parameters: bf16 for the kernels, fp32 master / m / v / grad for the optimizer
        self.params = []                      # dicts for lsp_adamw_step, in a fixed order
        self.layer_w, self.layer_g = [], []
        # gradient buckets (one flat buffer = one all-reduce each): the layers, then {head, final gain}, then the table
        lshapes = harness.WEIGHT_SHAPES(w)
        bshapes = [lshapes] * n_layers + [dict(head=(vocab, H), g_final=(H,)), dict(table=(vocab, H))]
        mult = 64 * world if zero1 else 64              # ZeRO-1 slices every flat bucket in `world` equal, 16-byte aligned parts
        self.buckets = dp.GradBuckets(bshapes, self.dev, group, multiple=mult)
        self.wbuckets = dp.GradBuckets(bshapes, self.dev, group, dtype=torch.bfloat16, multiple=mult)     # the bf16 weights, same layout
        self.world = world
        # fp16 tensor-core operand copies of every layer's projection weights (lsp_layer_weights.f16_cache): converted here
        # once; afterwards lsp_adamw_step writes them together with the bf16 weights (lsp_adamw_tensor.weight_f16), so no
        # forward pass of an iteration -- micro-batches, recomputation -- launches a weight cast
        self.caches = []
        for l in range(n_layers):
            bits = weights[l] if weights is not None else synth.layer_weights(w, l)
            for k, t in harness.upload_weights(bits, self.dev).items():
                self.wbuckets.views[l][k].copy_(t)
            cache = torch.empty(self.ctx.weight_cache_bytes, dtype=torch.uint8, device=self.dev)
            lw = dict(self.wbuckets.views[l])
            B.lsp_layer_prepare_weights(self.ctx, lw, cache)
            lw["f16_cache"] = cache
            self.caches.append(cache)
            self.layer_w.append(lw)
            self.layer_g.append(self.buckets.views[l])
        st = None
        if embedding is None or head is None:
            st = synth.stack_inputs(w.with_(vocab=vocab))
        self.table, self.w_head = self.wbuckets.views[n_layers + 1]["table"], self.wbuckets.views[n_layers]["head"]
        self.g_final = self.wbuckets.views[n_layers]["g_final"]
        self.table.copy_(harness.bf16_to_device(embedding if embedding is not None else st["embedding"], self.dev))
        self.w_head.copy_(harness.bf16_to_device(head if head is not None else synth.normal_bf16(w.cfg_id, 0, "w_head", (vocab, H), 0.02), self.dev))
        self.g_final.copy_(harness.bf16_to_device(g_final, self.dev) if g_final is not None
                           else torch.ones(H, dtype=torch.bfloat16, device=self.dev))
        self.d_head, self.d_gfinal = self.buckets.views[n_layers]["head"], self.buckets.views[n_layers]["g_final"]
        self.d_table = self.buckets.views[n_layers + 1]["table"]
        decay = [{k: len(s) == 2 for k, s in b.items()} for b in bshapes]
        self.zero = dp.Zero1State(self.buckets, self.wbuckets, decay, world, rank, group) if zero1 else None
        if not zero1:
            which = {k: i for i, k in enumerate(("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down"))}
            for b, shapes in enumerate(bshapes):
                for k in (synth.WEIGHT_NAMES if b < n_layers else shapes):
                    w16 = None
                    if b < n_layers and k in which:
                        off = B.lsp_weight_cache_offset(self.ctx, which[k])       # -1: rows permuted in the cache (rope_layout 1)
                        if off >= 0:
                            n = self.wbuckets.views[b][k].numel()
                            w16 = self.caches[b][off:off + 2 * n].view(torch.float16)
                    self._register(self.wbuckets.views[b][k], self.buckets.views[b][k], decay=decay[b][k], weight_f16=w16)
        self.t = 0
        # gradients are carried scaled by T (the gradient of the SUM loss): the mean's 1/T would push the layers' 16-bit
        # backward operands under the fp16 normal range; lsp_adamw_step divides it out (exact for a power-of-two T),
        # together with the number of replicas whose gradients were summed
        self.head_scale = float(T)
        self.grad_scale = dp.global_grad_scale(T * micro_batches, world)

    def _register(self, weight, grad, decay, weight_f16=None):
        self.params.append(dict(grad=grad, master=weight.float(), m=torch.zeros_like(grad), v=torch.zeros_like(grad), weight=weight,
                                decay=decay, weight_f16=weight_f16))

    @property
    def n_params(self):
        return sum(torch.Size(s).numel() for b in self.buckets.shapes for s in b.values())

    def forward_backward(self, ids: torch.Tensor, targets: torch.Tensor, stream=None, micro: int = 0):
        """ids, targets: int32 [T] on the device (micro-batch `micro` of n_micro).  Leaves the loss of the micro-batch in
        self.micro_losses[micro] (device) and every gradient in place; the all-reduces of the data-parallel replicas are
        issued during the last micro-batch's backward."""
        c, L = (self.ctx if micro == 0 else self.ctx_acc), self.L
        last = micro == self.n_micro - 1
        self.loss = self._loss_buf[micro, 0:1]
        B.lsp_embed_fwd(c, ids, self.table, self.xs[0], stream)
        for l in range(L):
            B.lsp_layer_fwd(c, self.xs[l], self.layer_w[l], self.xs[l + 1], self.saved[l], self.ws, stream)
        d_in = self.d[L & 1]
        B.lsp_head_fwd_bwd(c, self.xs[L], self.g_final, self.w_head, targets, self.V, self.loss, self.lse, d_in, self.d_gfinal,
                           self.d_head, self.ws, stream, grad_scale=self.head_scale)
        if last:
            self._reduce(L)
        for l in range(L - 1, -1, -1):
            d_out = self.d[l & 1]
            if self.recompute and l != L - 1:           # the shared buffer still holds the last layer's activations
                B.lsp_layer_fwd(c, self.xs[l], self.layer_w[l], self.xs[l + 1], self.saved[l], self.ws, stream)
            B.lsp_layer_bwd(c, self.xs[l], d_in, self.layer_w[l], self.saved[l], d_out, self.layer_g[l], self.ws, stream)
            if last:
                self._reduce(l)                     # overlaps the next layer's backward
            d_in = d_out
        B.lsp_embed_bwd(c, ids, d_in, self.V, self.d_table, stream)
        if last:
            self._reduce(L + 1)
        return self.loss

    def _reduce(self, b: int):
        """Exchange step of bucket b: all-reduce of the gradients, or reduce-scatter to their owners under ZeRO-1."""
        if self.zero is not None:
            self.zero.reduce_scatter_async(b)
        else:
            self.buckets.reduce_async(b)

    def optimizer_step(self, lr=None, stream=None, **hyper):
        self.t += 1
        lr = B.lsp_lr_cosine(self.t) if lr is None else lr
        if self.zero is not None:
            self.zero.step(lambda t, phase, gn: B.lsp_adamw_step(self.ctx, t, lr=lr, step=self.t, gnorm_out=gn, phase=phase,
                                                                 grad_scale=self.grad_scale, stream=stream, **hyper), self.gnorm)
            # the all-gathered bf16 weights came from other ranks' optimizer slices: refresh the operand caches from them
            for l in range(self.L):
                B.lsp_layer_prepare_weights(self.ctx, self.layer_w[l], self.caches[l], stream)
            return
        self.buckets.wait()
        B.lsp_adamw_step(self.ctx, self.params, lr=lr, step=self.t, gnorm_out=self.gnorm,
                         grad_scale=self.grad_scale, stream=stream, **hyper)

    def step(self, ids, targets, lr=None, stream=None, **hyper):
        """One iteration.  ids / targets: one [T] tensor each, or a list of n_micro of them (gradient accumulation)."""
        if isinstance(ids, torch.Tensor):
            ids, targets = [ids], [targets]
        assert len(ids) == self.n_micro == len(targets)
        for i, (a, b) in enumerate(zip(ids, targets)):
            self.forward_backward(a, b, stream, micro=i)
        self.optimizer_step(lr, stream, **hyper)
        return self.micro_losses

    def close(self):
        self.ctx.close()
        if self.ctx_acc is not None:
            self.ctx_acc.close()


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--layers", type=int, default=synth.CFG3_3B_STACK.n_layers)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=2)
    ap.add_argument("--zero1", action="store_true", help="optimizer state sharded over the data-parallel replicas (ZeRO stage 1)")
    ap.add_argument("--recompute", action="store_true", help="keep layer inputs only; re-run each layer's forward before its backward")
    args = ap.parse_args(argv)
    w = synth.CFG3_3B_STACK
    # under torchrun: data-parallel replicas, every rank takes a batch of the config's size (weak scaling) with its own ids
    renv = replicas.rank_env()
    if renv.world_size > 1:
        torch.cuda.set_device(renv.local_rank)
    dev = harness.require_cuda()
    replicas.init("nccl", renv)
    run = PretrainStep(w, args.layers, w.vocab, dev, world=renv.world_size, recompute=args.recompute, zero1=args.zero1, rank=renv.rank)
    s = synth.stack_inputs(w)
    ids = torch.from_numpy(s["ids"]).to(dev)
    ids = torch.roll(ids, 997 * renv.rank)
    targets = torch.roll(ids, -1)                     # next-token targets of the synthetic stream
    losses = []
    for _ in range(args.warmup):
        losses.append(float(run.step(ids, targets).cpu()))
    torch.cuda.synchronize()
    replicas.barrier(dev)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ms_fb = ms_opt = 0.0
    for _ in range(args.steps):
        e[0].record(); run.forward_backward(ids, targets)
        e[1].record(); run.optimizer_step()
        e[2].record(); torch.cuda.synchronize()
        ms_fb += e[0].elapsed_time(e[1]); ms_opt += e[1].elapsed_time(e[2])
        losses.append(float(run.loss.cpu()))
    ms_fb /= args.steps; ms_opt /= args.steps
    n = run.n_params
    tok_s, ms_it, tokens = replicas.whole_job_throughput(w.tokens, ms_fb + ms_opt, dev)      # all ranks' tokens / max time
    # the paper's accounting: 6 FLOPs per parameter per token without the embedding table, plus attention
    flops = renv.world_size * (6.0 * (n - w.vocab * w.hidden) * w.tokens + args.layers * 3.5 * synth.attn_flops_fwd(w, causal=True))
    if renv.is_main:
        print(json.dumps({"config": f"pretrain_{w.name}_L{args.layers}" + ("_recompute" if args.recompute else "") + ("_zero1" if args.zero1 else ""), "n_gpus": renv.world_size, "params": n, "tokens": int(tokens),
                          "ms_fwd_bwd": round(ms_fb, 3), "ms_adamw": round(ms_opt, 3), "ms_iteration": round(ms_it, 3),
                          "tokens_per_s": round(tok_s, 1), "model_tflops": round(flops / (ms_it * 1e-3) / 1e12, 1),
                          "adamw_GB_per_s": round(34.0 * n / (ms_opt * 1e-3) / 1e9, 1),
                          "mem_GB": round(torch.cuda.max_memory_allocated() / 1e9, 1), "loss": [round(x, 4) for x in losses]}))
    replicas.finalize()
    run.close()
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
