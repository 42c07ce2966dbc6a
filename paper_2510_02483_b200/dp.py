"""Data-parallel replicas: the batch is partitioned across ranks, sequences are
independent in the forward and backward pass, and the one exchange step of the path is the SUM of the weight / gain
gradients over ranks.  One process per GPU, torch.distributed for the plumbing (NCCL over NVLink 5 / NVSwitch on the
GPUs; the same code runs over gloo on CPU tensors, which is how the tests cover it).

`GradBuckets` lays the gradients of each bucket (one decoder layer, or the embedding / head tensors) out in ONE flat fp32
buffer, so a bucket is a single all-reduce (403 MB for the 3B-shape layer) that is issued as soon as the bucket's
backward has been enqueued and overlaps the backward of the next layer; `wait()` orders the optimizer step after all of
them.  No averaging pass exists: every rank carries its gradients scaled by its local token count T_local (section 13
of DESIGN.md), the sum over ranks is T_local * world * (gradient of the global mean loss), and that factor is handed to
lsp_adamw_step as grad_scale (`global_grad_scale`).  The sum runs in fp32 in the order the backend fixes.

UNMEASURED ON HARDWARE: rounds 1 and 2 had one GPU.  No NCCL rank has run this module; "overlaps the backward of the next
layer" describes how the calls are ordered (the collective is enqueued behind the bucket's backward and runs on the
backend's stream), not a timing that was taken.  Covered by the world_size-2 gloo tests of tests/test_dp_gloo.py only.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n_sequences: int, rank: int, world: int):
    """Contiguous block of sequences of rank `rank`: the first n % world ranks take one more."""
    base, extra = divmod(n_sequences, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def global_grad_scale(tokens_local: int, world: int) -> float:
    """grad_scale for lsp_adamw_step after the all-reduce, when every rank ran lsp_head_fwd_bwd with grad_scale =
    tokens_local (equal shards): stored sum = tokens_local * world * d(global mean loss)."""
    return float(tokens_local) * float(world)


def bucket_layout(shapes: dict, multiple: int = 64):
    """Offsets (in elements) of the tensors of a bucket inside its flat buffer, each on a 64-element boundary, and the
    flat length, padded to a multiple of `multiple` (itself a multiple of 64).  ZeRO-1 slices the flat buffer in `world`
    equal parts whose boundaries must stay on 4-element / 16-byte boundaries (lsp_adamw_step): use multiple = 64 * world
    (64 alone covers world = 1, 2, 4, 8, 16 only)."""
    assert multiple % 64 == 0
    offs, n = {}, 0
    for k, s in shapes.items():
        offs[k] = n
        n += (torch.Size(s).numel() + 63) // 64 * 64
    return offs, (n + multiple - 1) // multiple * multiple


class GradBuckets:
    def __init__(self, buckets, device, group=None, dtype=torch.float32, multiple: int = 64):
        """buckets: list of dicts name -> shape.  Allocates one flat buffer per bucket (fp32 for gradients; the same
        class lays out the bf16 weights for the sharded optimizer); `views[i][name]` are the tensors the kernels read or
        write (each starts on a 256-byte boundary for fp32: TMA stores, float4 loads).  multiple: see bucket_layout."""
        self.group = group
        self.shapes = list(buckets)
        self.multiple = multiple
        self.flat, self.views, self._pending = [], [], []
        for shapes in buckets:
            offs, n = bucket_layout(shapes, multiple)
            flat = torch.zeros(n, dtype=dtype, device=device)
            self.flat.append(flat)
            self.views.append({k: flat[offs[k]:offs[k] + torch.Size(s).numel()].view(s) for k, s in shapes.items()})

    def reduce_async(self, i: int):
        """All-reduce (sum) bucket i.  With NCCL the collective is ordered after the work already enqueued on the current
        stream and runs on the backend's own stream, so it overlaps what the caller enqueues next."""
        if dist.is_initialized() and dist.get_world_size(self.group) > 1:
            self._pending.append(dist.all_reduce(self.flat[i], op=dist.ReduceOp.SUM, group=self.group, async_op=True))

    def wait(self):
        """Order the current stream after every pending all-reduce (no host block with NCCL)."""
        for h in self._pending:
            h.wait()
        self._pending = []


def mean_loss(loss: torch.Tensor, group=None) -> torch.Tensor:
    """Mean over ranks of the per-rank mean loss (equal shards), in place."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(loss, op=dist.ReduceOp.SUM, group=group)
        loss /= dist.get_world_size(group)
    return loss


class Zero1State:
    """ZeRO stage 1: the model is replicated, the optimizer state is not.  Rank r owns the r-th 1/world of
    every gradient bucket: the bucket's gradient is reduce-scattered instead of all-reduced, the rank keeps fp32 master
    weights and moments for its slice only (12 bytes per parameter / world instead of 12), updates the slice, and the
    bf16 weights are all-gathered back into every replica's flat weight bucket.  The global gradient norm needs one
    scalar all-reduce between the two phases of the optimizer call (lsp_adamw_step phase 1 / 2).

    Device-agnostic: `step(phase_fn, ...)` takes the function that runs a phase on a list of tensor dicts -- the library
    call on the GPU, the fp64 oracle in the CPU tests."""

    def __init__(self, grads: GradBuckets, weights: GradBuckets, decay: list, world: int, rank: int, group=None):
        """grads / weights: buckets of identical layout (fp32 / bf16); decay: per bucket, dict name -> bool."""
        self.grads, self.weights, self.world, self.rank, self.group = grads, weights, world, rank, group
        self.lo, self.g_shard, self.master, self.m, self.v, self.segments = [], [], [], [], [], []
        self._pending = []
        assert grads.multiple == weights.multiple, "gradient and weight buckets must share one layout"
        for b, shapes in enumerate(grads.shapes):
            offs, n = bucket_layout(shapes, grads.multiple)
            if n % (4 * world):
                raise ValueError(f"ZeRO-1: bucket {b} has {n} elements, not a multiple of 4 * world = {4 * world}: the tail would "
                                 f"never be updated and slice boundaries would leave 16-byte alignment; build the buckets with "
                                 f"GradBuckets(..., multiple=64 * world)")
            per = n // world
            lo, hi = rank * per, (rank + 1) * per
            self.lo.append(lo)
            flat_g = grads.flat[b]
            self.g_shard.append(flat_g[lo:hi] if world == 1 else torch.zeros(per, dtype=flat_g.dtype, device=flat_g.device))
            self.master.append(weights.flat[b][lo:hi].float())
            self.m.append(torch.zeros(per, dtype=torch.float32, device=flat_g.device))
            self.v.append(torch.zeros(per, dtype=torch.float32, device=flat_g.device))
            segs = []
            for k, s in shapes.items():
                a, e = max(offs[k], lo), min(offs[k] + torch.Size(s).numel(), hi)
                if a < e:
                    segs.append((k, a, e, bool(decay[b][k])))
            self.segments.append(segs)

    def _native(self) -> bool:
        return dist.get_backend(self.group) != "gloo"       # gloo (CPU tests) has no reduce-scatter: emulate with all-reduce

    def reduce_scatter_async(self, b: int):
        if self.world > 1:
            if self._native():
                self._pending.append(dist.reduce_scatter_tensor(self.g_shard[b], self.grads.flat[b], op=dist.ReduceOp.SUM,
                                                                group=self.group, async_op=True))
            else:
                dist.all_reduce(self.grads.flat[b], op=dist.ReduceOp.SUM, group=self.group)
                per = self.g_shard[b].numel()
                self.g_shard[b].copy_(self.grads.flat[b][self.lo[b]:self.lo[b] + per])

    def tensors(self):
        """The tensor dicts of lsp_adamw_step for this rank's slices (a parameter cut by a slice boundary appears as the
        part this rank owns)."""
        out = []
        for b, segs in enumerate(self.segments):
            lo = self.lo[b]
            for _, a, e, dec in segs:
                out.append(dict(grad=self.g_shard[b][a - lo:e - lo], master=self.master[b][a - lo:e - lo], m=self.m[b][a - lo:e - lo],
                                v=self.v[b][a - lo:e - lo], weight=self.weights.flat[b][a:e], decay=dec))
        return out

    def step(self, phase_fn, sumsq: torch.Tensor):
        """phase_fn(tensors, phase, sumsq): phase 1 leaves this rank's sum of g^2 in sumsq[0]; phase 2 finds the global sum
        there and updates master / m / v / weight of the slices.  Then every replica gets all updated bf16 weights."""
        for h in self._pending:
            h.wait()
        self._pending = []
        t = self.tensors()
        phase_fn(t, 1, sumsq)
        if self.world > 1:
            dist.all_reduce(sumsq[0:1], op=dist.ReduceOp.SUM, group=self.group)
        phase_fn(t, 2, sumsq)
        if self.world > 1:
            for b in range(len(self.segments)):
                per = self.g_shard[b].numel()
                lo = self.lo[b]
                mine = self.weights.flat[b][lo:lo + per].clone()
                if self._native():
                    dist.all_gather_into_tensor(self.weights.flat[b], mine, group=self.group)
                else:
                    parts = [torch.empty_like(mine) for _ in range(self.world)]
                    dist.all_gather(parts, mine, group=self.group)
                    self.weights.flat[b].copy_(torch.cat(parts))
