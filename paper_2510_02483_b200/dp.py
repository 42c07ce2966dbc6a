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


class GradBuckets:
    def __init__(self, buckets, device, group=None):
        """buckets: list of dicts name -> shape.  Allocates one flat fp32 buffer per bucket; `views[i][name]` are the
        gradient tensors the backward writes into (each starts on a 256-byte boundary: TMA stores, float4 loads)."""
        self.group = group
        self.flat, self.views, self._pending = [], [], []
        for shapes in buckets:
            offs, n = {}, 0
            for k, s in shapes.items():
                offs[k] = n
                cnt = 1
                for d in s:
                    cnt *= d
                n += (cnt + 63) // 64 * 64
            flat = torch.zeros(n, dtype=torch.float32, device=device)
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
