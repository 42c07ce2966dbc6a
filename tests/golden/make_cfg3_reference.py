"""Writes tests/golden/cfg3_reference.npz: the compact fp64-oracle reference of BASELINE.json configs[2]
(28-layer 3B stack, batch 2 x seq 4096, vocab 128256) at its own size.

    python tests/golden/make_cfg3_reference.py [--out PATH] [--layers N]

Why a stored reference (decision rule for cfg 3): the oracle needs about
35 s per layer forward+backward on the GPU box's 16 host cores (plus one recomputed forward), i.e. 20-25 minutes for
the 28 layers -- it does not fit the 1200 s limit of the `-m gpu` suite.  So the reference is computed ONCE by this
script, which imports only `oracle/` and the seeded input generator (`synth.py`, no arithmetic of the method), and the
GPU test `test_stack_cfg3_full_depth_sampled` compares the CUDA path against it -- labelled "sampled", because the
file keeps, per tensor, its rms over ALL elements (the metric's denominator), a fixed seeded sample of elements and
the rows of largest reference norm, not every element.  The same comparison over every element runs on demand with
LSP_CFG3_FULL=1 (tests/test_gpu_parity.py::test_stack_cfg3_full_depth_every_element; log in profiles/).

No value in the file comes from the CUDA path.  Contents (float32 unless noted):
  y, dx0                 : "<name>/rms" (float64 scalar over the whole [T,H] tensor), "<name>/val" (the reference at
                           the flat indices sample_indices(...) -- regenerated from the seed, not stored),
                           "<name>/rows" (int64 row numbers of the rows of largest reference l2 norm), "<name>/rowval"
  L<l>/d<weight>         : the same four entries for each of the 7 projection-weight gradients of layer l
  L<l>/dg_attn, dg_mlp   : the full [H] gain gradients ("/full") and their rms
Sample seeds: numpy default_rng(SeedSequence([2510, 2483, 3, 7001, layer, tensor_id])) -- fixed here, before any
GPU result existed.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import lspref as R  # noqa: E402
from paper_2510_02483_b200 import synth  # noqa: E402  (seeded inputs only)

N_SAMPLE_ACT = 1 << 18      # sampled elements of y / dx0
N_ROWS_ACT = 16             # rows of largest reference norm of y / dx0
N_SAMPLE_W = 1 << 14        # sampled elements of every weight gradient
N_ROWS_W = 2                # rows of largest reference norm of every weight gradient
W2D = ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down")


def sample_rng(layer: int, tensor_id: int):
    return np.random.default_rng(np.random.SeedSequence([2510, 2483, 3, 7001, layer, tensor_id]))


def sample_indices(size: int, layer: int, tensor_id: int, n_sample: int) -> np.ndarray:
    """The fixed sample of flat element indices of a tensor of `size` elements (sorted, no repeats)."""
    return np.sort(sample_rng(layer, tensor_id).choice(size, size=min(n_sample, size), replace=False)).astype(np.int64)


# (layer, tensor_id, n_sample) of every sampled tensor, shared with the test that regenerates the indices
def sample_spec(name: str, layer: int = 0):
    if name == "y":
        return 0, 100, N_SAMPLE_ACT
    if name == "dx0":
        return 0, 101, N_SAMPLE_ACT
    return layer, synth.TENSOR_ID[name], N_SAMPLE_W


def compact(out: dict, key: str, ref: np.ndarray, layer: int, tensor_id: int, n_sample: int, n_rows: int):
    """rms over all elements, a seeded element sample, and the n_rows rows of largest l2 norm."""
    ref = np.asarray(ref, np.float64)
    flat = ref.reshape(-1)
    out[key + "/rms"] = np.float64(np.sqrt(np.mean(flat * flat)))
    idx = sample_indices(flat.size, layer, tensor_id, n_sample)
    out[key + "/val"] = flat[idx].astype(np.float32)
    norms = np.sqrt(np.sum(ref * ref, axis=1))
    rows = np.sort(np.argsort(norms)[-n_rows:])
    out[key + "/rows"] = rows.astype(np.int64)
    out[key + "/rowval"] = ref[rows].astype(np.float32)


class LazyWeights:
    """Sequence of the per-layer weight dicts (fp64), generated from the seeds on access: 28 layers of fp64 weights
    would be 22 GB.  `stack_fwd_bwd` only iterates, indexes and takes len()."""

    def __init__(self, w, n_layers):
        self.w, self.n = w, n_layers

    def __len__(self):
        return self.n

    def __getitem__(self, l):
        if not 0 <= l < self.n:
            raise IndexError(l)
        return {k: synth.bf16_bits_to_f64(v) for k, v in synth.layer_weights(self.w, l).items()}

    def __iter__(self):
        return (self[l] for l in range(self.n))


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg3_reference.npz"))
    ap.add_argument("--layers", type=int, default=0, help="depth (default: the workload's 28)")
    args = ap.parse_args(argv)
    w = synth.CFG3_3B_STACK
    n_layers = args.layers or w.n_layers
    cfg = R.LayerShape(w.batch, w.seq, w.hidden, w.n_q_heads, w.n_kv_heads, w.head_dim, w.ffn, w.rms_eps, w.rope_base)
    s = synth.stack_inputs(w)
    x0 = R.embed_fwd(s["ids"], synth.bf16_bits_to_f64(s["embedding"]))
    dy = synth.bf16_bits_to_f64(s["dy"])
    t0 = time.time()
    y, dx0, grads = R.stack_fwd_bwd(x0, dy, LazyWeights(w, n_layers), cfg)
    print(f"oracle stack_fwd_bwd, {n_layers} layers: {time.time() - t0:.0f} s", flush=True)
    out = {"n_layers": np.int64(n_layers)}
    compact(out, "y", y, 0, 100, N_SAMPLE_ACT, N_ROWS_ACT)
    compact(out, "dx0", dx0, 0, 101, N_SAMPLE_ACT, N_ROWS_ACT)
    for l in range(n_layers):
        for k in W2D:
            compact(out, f"L{l}/d{k}", grads[l][k], l, synth.TENSOR_ID[k], N_SAMPLE_W, N_ROWS_W)
        for k in ("g_attn", "g_mlp"):
            g = np.asarray(grads[l][k], np.float64)
            out[f"L{l}/d{k}/rms"] = np.float64(np.sqrt(np.mean(g * g)))
            out[f"L{l}/d{k}/full"] = g.astype(np.float32)
    np.savez(args.out, **out)
    print("wrote", args.out, os.path.getsize(args.out) // 1024, "KiB", flush=True)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
