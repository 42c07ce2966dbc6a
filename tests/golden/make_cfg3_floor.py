"""Writes tests/golden/cfg3_floor_<fmt>.json: the EMULATED-PRECISION FLOOR of BASELINE.json configs[2] (28-layer stack).

    python tests/golden/make_cfg3_floor.py [--fmt f16|bf16]

SURVEY.md 8(c) (last paragraph): where a tensor's error exceeds the 2e-2 bar, its emulated floor is reported beside the GPU
number -- the metric is not loosened.  The floor is the error of oracle/emulate16.py (float64 arithmetic, values rounded
to 16 bits only where a tensor-core implementation must feed 16-bit operands) against the exact oracle, in the same
per-tensor metric and at the same sampled positions as tests/golden/cfg3_reference.npz (max |emulated - ref| over the
sample and the largest-norm rows, divided by the reference rms over all elements).  Imports only oracle/ and the
seeded input generator; about 70 minutes on 8 cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import emulate16 as E  # noqa: E402
from oracle import lspref as R  # noqa: E402
from paper_2510_02483_b200 import synth  # noqa: E402
from tests.golden import make_cfg3_reference as M  # noqa: E402


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--fmt", default="f16", choices=["f16", "bf16"])
    args = ap.parse_args(argv)
    ref = np.load(os.path.join(HERE, "cfg3_reference.npz"))
    w = synth.CFG3_3B_STACK
    n_layers = int(ref["n_layers"])
    cfg = R.LayerShape(w.batch, w.seq, w.hidden, w.n_q_heads, w.n_kv_heads, w.head_dim, w.ffn, w.rms_eps, w.rope_base)
    s = synth.stack_inputs(w)
    x0 = R.embed_fwd(s["ids"], synth.bf16_bits_to_f64(s["embedding"]))
    dy = synth.bf16_bits_to_f64(s["dy"])
    floors = {}

    def err(key, name, layer, got):
        got = np.asarray(got, np.float64)
        idx = M.sample_indices(got.size, *M.sample_spec(name, layer))
        e = max(np.max(np.abs(got.reshape(-1)[idx] - ref[key + "/val"].astype(np.float64))),
                np.max(np.abs(got[ref[key + "/rows"]] - ref[key + "/rowval"].astype(np.float64))))
        floors[key] = float(e / float(ref[key + "/rms"]))

    def on_grads(l, g):
        for k in M.W2D:
            err(f"L{l}/d{k}", k, l, g[k])
        for k in ("g_attn", "g_mlp"):
            key = f"L{l}/d{k}"
            floors[key] = float(np.max(np.abs(g[k] - ref[key + "/full"].astype(np.float64))) / float(ref[key + "/rms"]))
        print(f"layer {l}: " + "  ".join(f"{k}={floors[f'L{l}/d{k}']:.2e}" for k in synth.WEIGHT_NAMES), flush=True)

    t0 = time.time()
    y, dx0, _ = E.stack_fwd_bwd(x0, dy, M.LazyWeights(w, n_layers), cfg, fmt=args.fmt, on_layer_grads=on_grads)
    err("y", "y", 0, y)
    err("dx0", "dx0", 0, dx0)
    print(f"emulated ({args.fmt}) stack: {time.time() - t0:.0f} s; y={floors['y']:.2e} dx0={floors['dx0']:.2e}", flush=True)
    out = os.path.join(HERE, f"cfg3_floor_{args.fmt}.json")
    with open(out, "w") as f:
        json.dump({"fmt": args.fmt, "n_layers": n_layers, "split_rows": 256, "floor": floors}, f, indent=0, sort_keys=True)
    print("wrote", out)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
