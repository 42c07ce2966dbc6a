"""Data-parallel path (paper_2510_02483_b200/dp.py) on CPU: two gloo ranks each run the fp64 oracle's
model forward+backward on their half of the batch, put their gradients -- scaled by the local token count, as
pretrain.PretrainStep carries them -- into GradBuckets, all-reduce, and must end with exactly what one process gets on
the whole batch once `global_grad_scale` is divided out (sequences are independent; only the weight gradients are sums
over tokens).  The CUDA kernels are not involved: this covers the host logic of the exchange step."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from tests.test_replicas_gloo import ROOT, free_port

WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["LSP_ROOT"])
import numpy as np, torch, torch.distributed as dist
from oracle import lspref as R, head_ref as Hd
from paper_2510_02483_b200 import dp
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
Bz, S, H, nq, nkv, d, F, V, L = 4, 16, 32, 2, 1, 16, 48, 40, 2
rng = np.random.default_rng(5)                      # same model and batch on every rank
names = ("wq", "wk", "wv", "wo", "g_attn", "w_gate", "w_up", "w_down", "g_mlp")
shapes = dict(wq=(nq * d, H), wk=(nkv * d, H), wv=(nkv * d, H), wo=(H, nq * d), g_attn=(H,), w_gate=(F, H), w_up=(F, H),
              w_down=(H, F), g_mlp=(H,))
layers = [{k: (1.0 + 0.1 * rng.standard_normal(s)) if k.startswith("g_") else 0.2 * rng.standard_normal(s) for k, s in shapes.items()}
          for _ in range(L)]
E, Wh, gf = 0.5 * rng.standard_normal((V, H)), 0.3 * rng.standard_normal((V, H)), 1.0 + 0.1 * rng.standard_normal(H)
ids = rng.integers(0, V, size=Bz * S); tg = rng.integers(0, V, size=Bz * S)

def model_grads(b0, b1):
    cfg = R.LayerShape(b1 - b0, S, H, nq, nkv, d, F, 1e-5, 10000.0, 0, True)
    i, y = ids[b0 * S:b1 * S], tg[b0 * S:b1 * S]
    xs, caches = [R.embed_fwd(i, E)], []
    for w in layers:
        o, c = R.layer_fwd(xs[-1], w, cfg); xs.append(o); caches.append(c)
    out = Hd.head_loss_fwd_bwd(xs[-1], gf, Wh, y, 1e-5)
    dd, lg = out["dx"], [None] * L
    for l in range(L - 1, -1, -1):
        dd, lg[l], _ = R.layer_bwd(dd, layers[l], cfg, caches[l])
    return out["loss"], lg, dict(head=out["dw_head"], g_final=out["dg_final"]), dict(table=Hd.embed_bwd(i, dd, V))

lo, hi = dp.shard_range(Bz, rank, world)
loss, lg, gh, gt = model_grads(lo, hi)
T_local = (hi - lo) * S
bk = dp.GradBuckets([shapes] * L + [dict(head=(V, H), g_final=(H,)), dict(table=(V, H))], "cpu")
for i, g in enumerate(lg + [gh, gt]):
    for k, v in g.items():
        bk.views[i][k].copy_(torch.from_numpy(v * T_local))      # fp32 buffers, as on the GPU
for i in range(L + 2):
    bk.reduce_async(i)
bk.wait()
scale = dp.global_grad_scale(T_local, world)
lt = dp.mean_loss(torch.tensor([loss], dtype=torch.float64))
full_loss, flg, fgh, fgt = model_grads(0, Bz)
worst = 0.0
for i, g in enumerate(flg + [fgh, fgt]):
    for k, v in g.items():
        got = bk.views[i][k].numpy().astype(np.float64) / scale
        worst = max(worst, float(np.max(np.abs(got - v)) / np.sqrt(np.mean(v * v))))
aligned = all((v.data_ptr() - f.data_ptr()) % 256 == 0 for f, b in zip(bk.flat, bk.views) for v in b.values())
print(json.dumps(dict(rank=rank, worst=worst, loss=float(lt), full_loss=full_loss, aligned=aligned, shard=[lo, hi])), flush=True)
dist.destroy_process_group()
"""


def test_shard_range_covers_batch():
    from paper_2510_02483_b200 import dp
    for n, world in ((8, 2), (7, 3), (2, 4), (256, 8)):
        r = [dp.shard_range(n, k, world) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
        sizes = [b - a for a, b in r]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    assert dp.global_grad_scale(8192, 8) == 65536.0


def test_grad_buckets_single_process_is_identity():
    import torch
    from paper_2510_02483_b200 import dp
    bk = dp.GradBuckets([dict(a=(3, 5), b=(7,)), dict(c=(2, 2))], "cpu")
    bk.views[0]["a"].fill_(2.0); bk.views[0]["b"].fill_(3.0); bk.views[1]["c"].fill_(4.0)
    bk.reduce_async(0); bk.reduce_async(1); bk.wait()
    assert float(bk.flat[0].sum()) == 2.0 * 15 + 3.0 * 7 and float(bk.flat[1].sum()) == 16.0
    assert bk.views[0]["b"].data_ptr() - bk.views[0]["a"].data_ptr() == 256          # 15 floats padded to 64


@pytest.mark.timeout(300)
def test_two_gloo_ranks_sum_to_full_batch_gradient():
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), LSP_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=280)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    assert sorted(tuple(o["shard"]) for o in outs) == [(0, 2), (2, 4)]
    for o in outs:
        assert o["aligned"]
        assert o["worst"] < 1e-6                                   # fp32 buffers: one rounding per addend
        assert o["loss"] == pytest.approx(o["full_loss"], rel=1e-12)


ZERO_WORKER = r"""
import json, os, sys
sys.path.insert(0, os.environ["LSP_ROOT"])
import numpy as np, torch, torch.distributed as dist
from oracle import adamw_ref as A
from paper_2510_02483_b200 import dp
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
shapes = [dict(wa=(24, 40), ga=(40,), wb=(40, 24)), dict(head=(50, 40), g_final=(40,)), dict(table=(50, 40))]
decay = [{k: len(s) == 2 for k, s in b.items()} for b in shapes]
rng = np.random.default_rng(11)                       # same initial weights everywhere
grads, weights = dp.GradBuckets(shapes, "cpu"), dp.GradBuckets(shapes, "cpu", dtype=torch.bfloat16)
for b in weights.views:
    for k, v in b.items():
        v.copy_(torch.from_numpy(0.05 * rng.standard_normal(tuple(v.shape))).to(torch.bfloat16))
w0 = [{k: v.float().numpy().astype(np.float64).copy() for k, v in b.items()} for b in weights.views]
T_local, scale = 16, dp.global_grad_scale(16, world)
def local_grads(r):                                   # what rank r's backward leaves in its buckets (scaled by T_local)
    g = np.random.default_rng(100 + r)
    return [{k: (3.0 * g.standard_normal(s) * T_local).astype(np.float32) for k, s in b.items()} for b in shapes]
mine = local_grads(rank)
for b, gb in enumerate(mine):
    for k, v in gb.items():
        grads.views[b][k].copy_(torch.from_numpy(v))
zero = dp.Zero1State(grads, weights, decay, world, rank)
lr, step = 1.0e-3, 1

def phase_fn(tensors, phase, sumsq):                  # the fp64 oracle in place of lsp_adamw_step
    if phase == 1:
        sumsq[0] = float(sum(float(np.sum(t["grad"].numpy().astype(np.float64) ** 2)) for t in tensors))
        return
    norm = float(np.sqrt(float(sumsq[0]))) / scale
    c = A.clip_coefficient(norm)
    for t in tensors:
        p, m, v, _ = A.adamw_step([t["master"].numpy()], [t["grad"].numpy().astype(np.float64) * (c / scale)], [t["m"].numpy()],
                                  [t["v"].numpy()], [t["decay"]], step, lr, clip=1e30)
        t["master"].copy_(torch.from_numpy(p[0])); t["m"].copy_(torch.from_numpy(m[0])); t["v"].copy_(torch.from_numpy(v[0]))
        t["weight"].copy_(torch.from_numpy(A.bf16_rne(t["master"].numpy())).to(torch.bfloat16))
    sumsq[0] = norm

for b in range(len(shapes)):
    zero.reduce_scatter_async(b)
sumsq = torch.zeros(2, dtype=torch.float32)
zero.step(phase_fn, sumsq)
# reference: one process, the summed gradients of both ranks, the whole model
tot = [{k: sum(local_grads(r)[b][k].astype(np.float64) for r in range(world)) / scale for k in shapes[b]} for b in range(len(shapes))]
names = [(b, k) for b in range(len(shapes)) for k in shapes[b]]
p_ref, _, _, norm_ref = A.adamw_step([w0[b][k] for b, k in names], [tot[b][k] for b, k in names], [np.zeros(shapes[b][k]) for b, k in names],
                                     [np.zeros(shapes[b][k]) for b, k in names], [decay[b][k] for b, k in names], step, lr)
worst, flips, n = 0.0, 0, 0
for (b, k), pr in zip(names, p_ref):
    got = weights.views[b][k].float().numpy().astype(np.float64)
    ref = A.bf16_rne(pr)
    flips += int(np.sum(got != ref)); n += got.size
    worst = max(worst, float(np.max(np.abs(got - pr) / (np.abs(pr) * 2.0 ** -8 + 1e-12))))
owned = sum(e - a for segs in zero.segments for _, a, e, _ in segs)
print(json.dumps(dict(rank=rank, norm=float(sumsq[0]), norm_ref=norm_ref, flips=flips, n=n, worst=worst, owned=owned)), flush=True)
dist.destroy_process_group()
"""


@pytest.mark.timeout(300)
def test_zero1_two_gloo_ranks_match_full_adamw():
    """dp.Zero1State over two gloo ranks with the fp64 oracle as the update function: reduce-scatter of the gradient
    buckets, sum of g^2 all-reduced between the two optimizer phases, slices updated by their owners, bf16 weights
    all-gathered -- every replica ends with the weights one process gets from AdamW on the summed gradients."""
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), LSP_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, "-c", ZERO_WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=280)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    total = sum(int(np.prod(s)) for b in [dict(wa=(24, 40), ga=(40,), wb=(40, 24)), dict(head=(50, 40), g_final=(40,)), dict(table=(50, 40))]
                for s in b.values())
    assert sum(o["owned"] for o in outs) == total                  # every parameter has exactly one owner
    for o in outs:
        assert o["norm"] == pytest.approx(o["norm_ref"], rel=1e-6)
        assert o["worst"] <= 1.01                                   # within half a bf16 ulp (+ fp32 master rounding) of the fp64 result
        assert o["flips"] <= 2e-3 * o["n"]                          # bf16 rounding of an fp32 vs an fp64 master weight


def test_zero1_slices_need_padded_buckets():
    """A world size that does not divide the 64-element padded bucket length (3, 6, ...) must not silently drop the tail of
    the flat buffer or cut slices off 16-byte boundaries: the constructor refuses, and buckets built with
    multiple = 64 * world give `world` equal slices that cover every parameter exactly once on 4-element boundaries."""
    import torch
    from paper_2510_02483_b200 import dp
    shapes = [dict(wa=(24, 40), ga=(40,), wb=(40, 24)), dict(table=(50, 40))]
    decay = [{k: len(s) == 2 for k, s in b.items()} for b in shapes]
    g, w = dp.GradBuckets(shapes, "cpu"), dp.GradBuckets(shapes, "cpu", dtype=torch.bfloat16)
    with pytest.raises(ValueError, match="multiple of 4 \\* world"):
        dp.Zero1State(g, w, decay, 3, 0)
    g3, w3 = dp.GradBuckets(shapes, "cpu", multiple=192), dp.GradBuckets(shapes, "cpu", dtype=torch.bfloat16, multiple=192)
    covered = [torch.zeros_like(f, dtype=torch.int32) for f in g3.flat]
    for r in range(3):
        z = dp.Zero1State(g3, w3, decay, 3, r)
        for b, segs in enumerate(z.segments):
            assert z.lo[b] % 4 == 0 and g3.flat[b].numel() % 3 == 0
            for _, a, e, _ in segs:
                assert a % 4 == 0 and e % 4 == 0
                covered[b][a:e] += 1
    for b, shp in enumerate(shapes):
        offs, _ = dp.bucket_layout(shp, 192)
        for k, s in shp.items():
            n = torch.Size(s).numel()
            assert bool((covered[b][offs[k]:offs[k] + n] == 1).all()), (b, k)
