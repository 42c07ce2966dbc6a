#!/usr/bin/env python
"""clock64 traces of the three tcgen05 attention kernels (forward, dK/dV, dQ) at the attention shape of config 2, and
(--gemm) the wait counters of the GEMM kernel's MMA warp for the 12 GEMM shapes of the config-2 step.

    python bench_trace.py [--blocks N] [--gemm] > profiles/rX_attn_traces.txt

Builds a DEBUG copy of the library with -DLSP_ATTN_TRACE into a temporary directory (the shipped liblsp.so carries no
trace code), loads it in place of the product library for this process only, runs lsp_sdpa_fwd / lsp_sdpa_bwd on the
seeded inputs of 4 sequences x 4096 tokens, 24 q / 8 kv heads, and prints, for consecutive key blocks of ONE CTA in its
steady state, the SM clock at which each pipeline event happened (relative to the first): when a softmax warp saw its
accumulator, finished its phase, when the MMA warp saw the operand and had issued each MMA group.  The per-block period
against the tensor cycles of a block (forward 2048 per tile pair, dK/dV 2048, dQ 768) is the kernel's tensor
utilisation in steady state; the gaps between events say where the rest goes.  A measurement aid:
it changes no result and is not part of the C ABI of include/lsp.h.
"""
from __future__ import annotations

import argparse
import ctypes as C
import os
import subprocess
import sys
import tempfile

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def build_traced(tmp):
    from paper_2510_02483_b200 import build as Bd
    out = os.path.join(tmp, "liblsp_trace.so")
    cmd = [os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")] + Bd.NVCC_FLAGS + ["-DLSP_ATTN_TRACE", "-DLSP_GEMM_TRACE", "-o", out] + Bd.SOURCES
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    return out


def table(a, names, nblocks):
    base = min(int(a[0, k]) for k in names if a[0, k])
    print("block  " + "  ".join(f"{names[k]:>12s}" for k in sorted(names)))
    for b in range(nblocks):
        print(f"{b:5d}  " + "  ".join(f"{(int(a[b, k]) - base) if a[b, k] else -1:12d}" for k in sorted(names)))
    first = sorted(names)[0]
    per = [(int(a[b + 1, first]) - int(a[b, first])) for b in range(nblocks - 1) if a[b, first] and a[b + 1, first]]
    per = sorted(p for p in per if p > 0)
    if per:
        print(f"median period between blocks: {per[len(per) // 2]} cycles")


def gemm_table(lib, B, harness, synth, torch, np):
    """Per GEMM shape of the cfg2 step (lsp_gemm, plain fp32 store): what the MMA-issuing warp of a CTA pair did -- cycles in its
    loop, share of them spent waiting for operand stages (it runs ahead of the tensor queue: a large share is normal) and for a
    free accumulator, and cycles per 64-wide k-block against the 512 tensor cycles a 256 x 256 x 64 pair step takes."""
    import bench_configs as BC
    lib.lsp_debug_read_gemm_trace.argtypes = [C.c_void_p, C.c_int]
    lib.lsp_debug_read_gemm_trace.restype = C.c_int
    dev = torch.device("cuda")
    ctx = harness.make_ctx(synth.CFG1_TINY)
    buf = (C.c_longlong * (128 * 4))()
    print("\n== gemm_pair_tcgen05_kernel, MMA warp of every CTA pair (mean over the pairs); 512 tensor cycles per k-block")
    print(f"{'stage':14s} {'M':>6s} {'N':>6s} {'K':>6s} {'ms':>7s} {'loop cycles':>12s} {'wait stages %':>14s} {'wait accum %':>13s} {'k-blocks':>9s} {'cycles/k-block':>15s} {'SM GHz':>7s}")
    for name, op, M, N, K in BC.gemm_shapes(synth.CFG2_3B_LAYER):
        a_shape = (K, M) if op == 2 else (M, K)
        b_shape = (N, K) if op == 0 else (K, N)
        a = torch.randn(a_shape, device=dev).to(torch.float16)
        b = torch.randn(b_shape, device=dev).to(torch.float16)
        c = torch.empty((M, N), dtype=torch.float32, device=dev)
        ms = BC._time(lambda: B.lsp_gemm(ctx, op, M, N, K, a, a_shape[1], B.LSP_F16, b, b_shape[1], B.LSP_F16, c, N), 20)
        assert lib.lsp_debug_read_gemm_trace(buf, 128 * 4) == 0
        t = np.array(buf[:], dtype=np.int64).reshape(128, 4)
        t = t[t[:, 3] > 0]
        loop = t[:, 0].astype(float)
        print(f"{name:14s} {M:6d} {N:6d} {K:6d} {ms:7.3f} {loop.mean():12.0f} {100 * t[:, 1].sum() / loop.sum():14.1f} "
              f"{100 * t[:, 2].sum() / loop.sum():13.1f} {t[:, 3].mean():9.0f} {(loop / t[:, 3]).mean():15.1f} {loop.max() / ms / 1e6:7.2f}")
        del a, b, c
    ctx.close()


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--blocks", type=int, default=24)
    ap.add_argument("--gemm", action="store_true", help="also print the GEMM kernel's MMA-warp wait counters per shape")
    args = ap.parse_args(argv)
    import numpy as np
    import torch
    from paper_2510_02483_b200 import binding as B
    from paper_2510_02483_b200 import harness, synth
    if not torch.cuda.is_available():
        raise B.LspError("bench_trace.py needs a CUDA device")
    with tempfile.TemporaryDirectory() as tmp:
        B.LIB_PATH = build_traced(tmp)                     # this process only; the product library is untouched
        lib = B.lib()
        lib.lsp_debug_read_trace.argtypes = [C.c_void_p, C.c_int]
        lib.lsp_debug_read_trace.restype = C.c_int
        w = synth.CFG5_ATTN[1].with_(batch=4)              # B 4 x S 4096, 24 q / 8 kv heads: the attention of config 2
        ctx = harness.make_ctx(w, use_rope=False)
        dev = torch.device("cuda")
        t = {k: harness.bf16_to_device(v, dev) for k, v in synth.attn_inputs(w).items()}
        Bz, S, nq, nkv, d = w.batch, w.seq, w.n_q_heads, w.n_kv_heads, w.head_dim
        o = torch.empty((Bz, S, nq, d), dtype=torch.float32, device=dev)
        lse = torch.empty((Bz, nq, S), dtype=torch.float32, device=dev)
        dq = torch.empty_like(o)
        dk = torch.empty((Bz, S, nkv, d), dtype=torch.float32, device=dev)
        dv = torch.empty_like(dk)
        ws = torch.empty(ctx.workspace_bytes, dtype=torch.uint8, device=dev)
        buf = (C.c_ulonglong * (64 * 32))()

        def read():
            assert lib.lsp_debug_read_trace(buf, 64 * 32) == 0
            return np.array(buf[:], dtype=np.uint64).reshape(64, 32)

        for _ in range(3):
            B.lsp_sdpa_fwd(ctx, t["q"], t["k"], t["v"], o, lse, ws)
        torch.cuda.synchronize()
        print("== attn_fwd_tc_kernel, CTA 3, key blocks 64.. of the CTA (tile 0 | tile 1 | MMA warp); 2048 tensor cycles per block and tile pair")
        table(read(), {0: "t0 s_full", 1: "t0 loaded", 2: "t0 max", 3: "t0 P part 0", 4: "t0 P part 1", 8: "t1 s_full", 12: "t1 arrive",
                       16: "mma P0", 17: "mma PV0", 19: "mma S0", 20: "mma P1", 21: "mma PV1", 23: "mma S1"}, args.blocks)
        for _ in range(3):
            B.lsp_sdpa_bwd(ctx, t["q"], t["k"], t["v"], o, lse, t["dO"], dq, dk, dv, ws)
        torch.cuda.synchronize()
        a = read()
        print("\n== attn_bwd_dkdv_tc_kernel, CTA 5, blocks 16.. (softmax warp | MMA warp); 2048 tensor cycles per 128 x 128 block")
        table(a, {0: "st_full", 1: "P arrive", 2: "dpt_full", 3: "dS arrive", 16: "mma P", 17: "dV issued", 18: "ST+1 issued", 19: "mma dS",
                  20: "dK issued", 21: "dPT+1 issued"}, args.blocks)
        print("\n== attn_bwd_dkdv_tc_kernel, lifetime of two CTAs (cycles from CTA entry): first S^T landed | last dS^T handed over | accumulators "
              "complete | stores written | exit   (block iterations)")
        for row, what in ((62, "heaviest key block (CTA 5)"), (63, "a light key block (CTA 900)")):
            t0 = int(a[row, 10])
            if t0:
                print(f"{what:32s}" + "  ".join(f"{int(a[row, k]) - t0:10d}" for k in range(11, 16)) + f"   ({int(a[row, 22])} iterations)")
        print("\n== attn_bwd_dq_tc_kernel, CTA 7, blocks 96.. (softmax warp | MMA warp); 768 tensor cycles per 128 x 64 block")
        table(a, {8: "sdp_full", 9: "dS arrive", 24: "mma dS", 25: "dQ issued", 26: "SdP+2 issued"}, args.blocks)
        ctx.close()
        if args.gemm:
            gemm_table(lib, B, harness, synth, torch, np)
        del lib
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
