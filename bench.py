#!/usr/bin/env python
"""bench.py -- BASELINE.json metric: "3B-shape layer fwd+bwd tokens/s; TFLOP/s as % of B200 dense BF16 peak".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg4|cfg1] [--impl ours|reference]

One step = one pass of the whole hot path (SURVEY.md 8(a) F1-F7 + B1-B10): lsp_layer_fwd + lsp_layer_bwd on
the seeded synthetic inputs of BASELINE.json configs[1] (single 3B-shape Llama decoder layer, batch 4 x seq 4096,
T = 16384 tokens).  `value` = tokens/s with inputs resident in HBM; `e2e` = the same through
lsp_layer_step_host with pinned HOST buffers (H2D of x, dy and D2H of y, dx inside the timed region).
N > 1: "replicas only" (north_star: no sharding, no collective) -- every rank runs the same step on its own
GPU, barrier + max-over-ranks device time, value = N*T / t  (weak scaling).
`--impl reference` times the fp64 CPU oracle (oracle/lspref.py, as it stands) on a bounded sample; the `cpu_baseline`
of our own line is ONE FULL step of the workload through the same oracle (about a minute on the box's 16 cores).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "3B-shape layer fwd+bwd tokens/s; TFLOP/s as % of B200 dense BF16 peak"
NOMINAL_BF16_TF = 2250.0            # B200 dense bf16, /opt/skills/guides/B200_PROFILING.md (nominal table)
FALLBACK_PEAKS = dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0)   # same guide, "fallback"
GEMM_STAGES = ("gemm_qkv_rope", "gemm_oproj_res", "gemm_gateup_swiglu", "gemm_down_res", "wgrad_down",
               "dgrad_down_swiglu_bwd", "wgrad_gateup", "dgrad_gateup", "wgrad_oproj", "dgrad_oproj", "wgrad_qkv",
               "dgrad_qkv")
# bounded oracle sample: the first SAMPLE_SEQ positions of ONE sequence of the workload (same H, heads, F)
SAMPLE_SEQ = 1024


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d["bf16_tflops"]),
                        bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"]))), "measured"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback"


def pick_workload(name):
    from paper_2510_02483_b200 import synth
    return {"cfg1": synth.CFG1_TINY, "cfg2": synth.CFG2_3B_LAYER, "cfg4": synth.CFG4_30B_LAYER}[name]


# --------------------------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event (throttle) reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                try:
                    bits = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    bits = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for b, n in self.REASONS.items():
                    if bits & b:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2.0)
        s = sorted(self.samples)
        return dict(sm_mhz=(s[len(s) // 2] if s else None), sm_max_mhz=self.max_mhz, reasons=sorted(self.reasons),
                    samples=len(s), power_w_max=(max(self.power) if self.power else None))


def physical_gpu_index(local_index):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_index])
        except Exception:
            return local_index
    return local_index


# --------------------------------------------------------------------------------------------- oracle legs
def oracle_sample_step(w, sample_seq):
    """Build the bounded oracle sample (first `sample_seq` positions of one sequence) and return a step closure."""
    import numpy as np
    from oracle import lspref as R
    from paper_2510_02483_b200 import synth
    S = min(sample_seq, w.seq)
    ws = w.with_(batch=1, seq=S)
    cfg = R.LayerShape(1, S, w.hidden, w.n_q_heads, w.n_kv_heads, w.head_dim, w.ffn, w.rms_eps, w.rope_base, 0, True)
    wt = {k: synth.bf16_bits_to_f64(v) for k, v in synth.layer_weights(w).items()}
    inp = synth.layer_inputs(ws)
    x, dy = synth.bf16_bits_to_f64(inp["x"]), synth.bf16_bits_to_f64(inp["dy"])

    def step():
        out = R.layer_fwd_bwd(x, dy, wt, cfg)
        return float(np.sum(out["y"][0, :4]))
    return step, S


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [int(p.get("num_threads", 0)) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return max(n)
    except Exception:
        pass
    return os.cpu_count() or 1


def time_oracle(w, steps, warmup, sample_seq=SAMPLE_SEQ):
    step, S = oracle_sample_step(w, sample_seq)
    for _ in range(warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = (time.perf_counter() - t0) / max(steps, 1)
    sample = (f"first {S} positions of 1 of {w.batch} sequences of {w.name} (T={S} tokens, full H/heads/FFN), "
              f"fp64 numpy oracle layer fwd+bwd, {steps} step(s); causal attention work per token is {S}/{w.seq} of the "
              f"full configuration's, the GEMM work per token is the same")
    return S / dt, dt, sample


def host_cpu():
    """(nproc, CPU model string) of the box the oracle is timed on (print both beside the baseline)."""
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.lower().startswith("model name"):
                    model = ln.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return os.cpu_count() or 0, model


def time_oracle_full(w):
    """One step of the WHOLE workload (every sequence, full length) through oracle/lspref.layer_fwd_bwd, as it stands."""
    from oracle import lspref as R
    from paper_2510_02483_b200 import synth
    cfg = R.LayerShape(w.batch, w.seq, w.hidden, w.n_q_heads, w.n_kv_heads, w.head_dim, w.ffn, w.rms_eps, w.rope_base, 0, True)
    wt = {k: synth.bf16_bits_to_f64(v) for k, v in synth.layer_weights(w).items()}
    inp = synth.layer_inputs(w)
    x, dy = synth.bf16_bits_to_f64(inp["x"]), synth.bf16_bits_to_f64(inp["dy"])
    t0 = time.perf_counter()
    R.layer_fwd_bwd(x, dy, wt, cfg)
    dt = time.perf_counter() - t0
    sample = (f"one full step of {w.name} (all {w.batch} sequences x {w.seq} positions, T={w.tokens}), fp64 numpy oracle "
              f"layer fwd+bwd, no warm-up")
    return w.tokens / dt, dt, sample


def run_reference(args):
    from paper_2510_02483_b200 import replicas
    renv = replicas.rank_env()
    if renv.rank != 0:
        return 0                                     # rank 0 alone runs and prints the reference arm
    w = pick_workload(args.workload)
    tps, dt, sample = time_oracle(w, args.steps, args.warmup)
    cores = blas_threads()
    line = {"impl": "reference", "metric": METRIC, "value": tps, "unit": "tokens/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "batch": w.batch, "seq": w.seq, "hidden": w.hidden, "n_q_heads": w.n_q_heads,
                       "n_kv_heads": w.n_kv_heads, "head_dim": w.head_dim, "ffn": w.ffn, "sample": sample},
            "cpu_baseline": {"value": tps, "unit": "tokens/s", "cores": cores, "kind": "oracle", "sample": sample,
                             "nproc": host_cpu()[0], "cpu_model": host_cpu()[1]},
            "e2e": {"value": tps, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    from paper_2510_02483_b200 import binding as B
    from paper_2510_02483_b200 import harness, replicas, synth

    renv = replicas.rank_env()
    if not torch.cuda.is_available():
        raise B.LspError("bench.py needs a CUDA device: the product path has no CPU fallback")
    B.lib()                                           # fail loudly when liblsp.so is missing
    torch.cuda.set_device(renv.local_rank % torch.cuda.device_count())
    dev = torch.device("cuda", torch.cuda.current_device())
    replicas.init("nccl", renv)

    w = pick_workload(args.workload)
    K, W = args.steps, max(args.warmup, 3)
    peaks, peak_src = load_peaks()

    ctx = harness.make_ctx(w)
    buf = harness.LayerBuffers(ctx, w, dev)
    weights = harness.upload_weights(synth.layer_weights(w), dev)
    inp = synth.layer_inputs(w)
    x, dy = harness.bf16_to_device(inp["x"], dev), harness.bf16_to_device(inp["dy"], dev)
    stream = torch.cuda.current_stream()
    # The weights do not change between the steps of this benchmark (no optimizer step in the metric), so their fp16
    # tensor-core operand copies are made ONCE, outside the timed region (lsp_layer_prepare_weights; in a training
    # iteration lsp_adamw_step writes them as part of the weight update).  --recast-weights times the other mode of the
    # same entry points: every forward converts the bf16 weights itself.
    if not args.recast_weights:
        weights = harness.with_weight_cache(ctx, weights, dev, stream)

    def step():
        B.lsp_layer_fwd(ctx, x, weights, buf.y, buf.saved, buf.ws, stream)
        B.lsp_layer_bwd(ctx, x, dy, weights, buf.saved, buf.dx, buf.grads, buf.ws, stream)

    for _ in range(W):
        step()
    torch.cuda.synchronize()

    # ------------------------------------------------------------------ timed region (device-resident inputs)
    sampler = ClockSampler(physical_gpu_index(dev.index))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier(dev)
    torch.cuda.synchronize()
    l0 = B.lsp_launch_count(ctx)
    sampler.start()
    e0.record(stream)
    for _ in range(K):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    replicas.barrier(dev)
    launches = B.lsp_launch_count(ctx) - l0
    ms_local = e0.elapsed_time(e1)
    value, ms_max, units = replicas.whole_job_throughput(float(w.tokens) * K, ms_local, dev)
    ms_step = ms_max / K

    # ------------------------------------------------------------------ end to end through host buffers
    # Every step uploads its x, dy from pinned host memory and downloads its y, dx (lsp_layer_step_host_async: the copies
    # of neighbouring steps overlap the compute; two device staging sets alternate); the timed region ends after the last
    # download (lsp_host_copies_wait + event).
    n = w.tokens * w.hidden
    hx, hdy = harness.bf16_pinned(inp["x"]), harness.bf16_pinned(inp["dy"])
    hy = torch.empty((w.tokens, w.hidden), dtype=torch.float32).pin_memory()
    hdx = torch.empty((w.tokens, w.hidden), dtype=torch.float32).pin_memory()
    x_st, dy_st = [torch.empty_like(x) for _ in range(2)], [torch.empty_like(dy) for _ in range(2)]
    y_st, dx_st = [buf.y, torch.empty_like(buf.y)], [buf.dx, torch.empty_like(buf.dx)]

    def steps_host(k):
        for i in range(k):
            B.lsp_layer_step_host_async(ctx, hx, hdy, weights, hy, hdx, buf.grads, x_st[i & 1], dy_st[i & 1], y_st[i & 1], dx_st[i & 1],
                                        buf.saved, buf.ws, stream)
        B.lsp_host_copies_wait(ctx, stream)

    # as many steps as the device-resident region: a shorter burst runs at a higher SM clock under the power cap and would
    # read faster than `value` (r1g: 10 host steps at 1.61 M tokens/s beside 50 resident steps at 1.59 M)
    Ke = max(3, K)
    steps_host(2)
    torch.cuda.synchronize()
    replicas.barrier(dev)
    e0.record(stream)
    steps_host(Ke)
    e1.record(stream)
    torch.cuda.synchronize()
    replicas.barrier(dev)
    e2e_value, _, _ = replicas.whole_job_throughput(float(w.tokens) * Ke, e0.elapsed_time(e1), dev)
    h2d, d2h = 2 * n * 2, 2 * n * 4

    # ------------------------------------------------------------------ per-step distribution, forward and backward apart
    # (SURVEY.md 8(d) timing protocol: median / min / p90; a separate pass, the headline above is the bracketed K steps)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K + 1)]
    ev[0].record(stream)
    for i in range(K):
        B.lsp_layer_fwd(ctx, x, weights, buf.y, buf.saved, buf.ws, stream)
        ev[2 * i + 1].record(stream)
        B.lsp_layer_bwd(ctx, x, dy, weights, buf.saved, buf.dx, buf.grads, buf.ws, stream)
        ev[2 * i + 2].record(stream)
    torch.cuda.synchronize()
    fwd_ms = sorted(ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(K))
    bwd_ms = sorted(ev[2 * i + 1].elapsed_time(ev[2 * i + 2]) for i in range(K))
    tot_ms = sorted(ev[2 * i].elapsed_time(ev[2 * i + 2]) for i in range(K))
    pick = lambda v, q: v[min(len(v) - 1, int(q * len(v)))]
    per_step = {"median": round(pick(tot_ms, 0.5), 4), "min": round(tot_ms[0], 4), "p90": round(pick(tot_ms, 0.9), 4),
                "fwd_median": round(pick(fwd_ms, 0.5), 4), "bwd_median": round(pick(bwd_ms, 0.5), 4)}

    # ------------------------------------------------------------------ per-stage device times (roofline of the GEMM kernel)
    B.lsp_timing_enable(ctx, K * 64)
    for _ in range(K):
        step()
    torch.cuda.synchronize()
    stages = B.lsp_timing_read(ctx)
    B.lsp_timing_enable(ctx, 0)
    stage_ms = {k: v[0] / K for k, v in stages.items()}
    gemm_ms = sum(stage_ms.get(s, 0.0) for s in GEMM_STAGES)
    gemm_launches = sum(stages[s][1] for s in GEMM_STAGES if s in stages) / K
    T, H, F = w.tokens, w.hidden, w.ffn
    nqd, nkvd = w.n_q_heads * w.head_dim, w.n_kv_heads * w.head_dim
    gemm_flops = 3.0 * 2.0 * T * (H * (nqd + 2 * nkvd) + nqd * H + 3 * H * F)
    flops = synth.layer_flops(w, causal=True)
    gemm_tf = gemm_flops / (gemm_ms * 1e-3) / 1e12 if gemm_ms > 0 else 0.0
    tflops = flops / (ms_step * 1e-3) / 1e12 * renv.world_size
    peak_t = peaks["bf16_tflops_sustained"]
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "gemm_traffic.json")      # written from an ncu --set full capture, if any
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(w.name)
        except Exception:
            traffic = None
    roofline = {"bound": "tensor", "kernel": "gemm_pair_tcgen05_kernel (12 GEMM launches of the step)",
                "achieved": gemm_tf, "peak": peak_t, "unit": "TFLOP/s", "frac": gemm_tf / peak_t,
                "peak_source": f"{peak_src} sustained cuBLAS bf16 (kernel timed inside a long step)",
                "traffic": traffic, "flops_per_step": gemm_flops, "ms_per_step": gemm_ms,
                "launches_per_step": gemm_launches, "share_of_step": gemm_ms / sum(stage_ms.values()) if stage_ms else None,
                "stage_ms": {k: round(v, 4) for k, v in sorted(stage_ms.items(), key=lambda kv: -kv[1])}}
    # The per-stage events of the timing pass sit BETWEEN the kernels: they add their own cost and cut the programmatic
    # dependent launches, so the stage times sum to more than the timed step.  Beside the event-measured figure above (the
    # one `frac` is built on), the same share applied to the untimed step: what the 12 GEMMs cost inside the step that `value` times.
    if stage_ms and sum(stage_ms.values()) > 0:
        in_step_ms = ms_step * gemm_ms / sum(stage_ms.values())
        roofline["in_untimed_step"] = {"ms_per_step": in_step_ms, "achieved": gemm_flops / (in_step_ms * 1e-3) / 1e12,
                                       "frac": gemm_flops / (in_step_ms * 1e-3) / 1e12 / peak_t,
                                       "how": "share_of_step x ms_per_step of the timed (event-free) loop"}

    # the kernel family FURTHEST from the tensor roof, beside the dominant one: causal attention forward + backward
    # (algorithmic FLOPs: 4 d nq S (S+1)/2 per sequence forward, x 2.5 backward; the recomputed S / dP of the backward
    # are not counted).  tensor_pipe_pct: from the committed ncu capture of the same step (profiles/attn_pipes.json).
    attn_stage_names = ("attn_fwd", "attn_bwd", "attn_bwd_dq", "attn_dvec")
    attn_ms = {k: stage_ms.get(k, 0.0) for k in attn_stage_names if k in stage_ms}
    attn_flops_fwd = synth.attn_flops_fwd(w, causal=True)
    attn_total_ms = sum(attn_ms.values())
    pipes = None
    ppath = os.path.join(ROOT, "profiles", "attn_pipes.json")
    if os.path.exists(ppath):
        try:
            pipes = json.load(open(ppath)).get(w.name)
        except Exception:
            pipes = None
    fwd_tf = attn_flops_fwd / (attn_ms.get("attn_fwd", 0.0) * 1e-3) / 1e12 if attn_ms.get("attn_fwd") else None
    bwd_ms = attn_total_ms - attn_ms.get("attn_fwd", 0.0)
    bwd_tf = 2.5 * attn_flops_fwd / (bwd_ms * 1e-3) / 1e12 if bwd_ms > 0 else None
    attn_tf = 3.5 * attn_flops_fwd / (attn_total_ms * 1e-3) / 1e12 if attn_total_ms > 0 else None
    roofline["kernels"] = [
        {"kernel": "gemm_pair_tcgen05_kernel x12", "bound": "tensor", "flops": gemm_flops, "ms": gemm_ms, "achieved": gemm_tf,
         "frac": gemm_tf / peak_t, "frac_of_nominal": gemm_tf / NOMINAL_BF16_TF, "frac_of_burst": gemm_tf / peaks["bf16_tflops"]},
        {"kernel": "attention family (attn_fwd_tc_kernel, attn_bwd_dkdv_tc_kernel, attn_bwd_dq_tc_kernel)", "bound": "tensor",
         "flops": 3.5 * attn_flops_fwd, "ms": attn_total_ms, "stage_ms": {k: round(v, 4) for k, v in attn_ms.items()},
         "achieved": attn_tf, "achieved_fwd": fwd_tf, "achieved_bwd": bwd_tf,
         "frac": (attn_tf / peak_t) if attn_tf else None, "frac_of_nominal": (attn_tf / NOMINAL_BF16_TF) if attn_tf else None,
         "frac_of_burst": (attn_tf / peaks["bf16_tflops"]) if attn_tf else None, "unit": "TFLOP/s", "peak": peak_t,
         "tensor_pipe_pct": pipes}]

    line = {"metric": METRIC, "value": value, "unit": "tokens/s", "n_gpus": renv.world_size, "steps": K, "warmup": W,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16/bf16 operands, f32 accumulate", "data": "synthetic",
            "config": {"workload": w.name, "batch": w.batch, "seq": w.seq, "hidden": w.hidden, "n_q_heads": w.n_q_heads,
                       "n_kv_heads": w.n_kv_heads, "head_dim": w.head_dim, "ffn": w.ffn, "parallelism": f"replicas x{renv.world_size}",
                       "l2": "working set (saved+ws+weights+grads > 3 GB) far exceeds the 126 MB L2; no flush needed",
                       "weights": ("bf16 weights re-converted to fp16 operands inside every forward" if args.recast_weights else
                                   "unchanged between steps: fp16 operand cache made once before the loop (lsp_layer_prepare_weights)"),
                       "launch": ("ordinary stream-ordered launches (LSP_PDL=0)" if os.environ.get("LSP_PDL") == "0" else
                                  "programmatic dependent launch between the kernels of a step (default; LSP_PDL=0 disables)")},
            "tflops": tflops, "flops_per_step": flops,
            "frac_of_nominal_bf16_peak": tflops / renv.world_size / NOMINAL_BF16_TF,
            "frac_of_measured_sustained": tflops / renv.world_size / peaks["bf16_tflops_sustained"],
            "frac_of_measured_burst": tflops / renv.world_size / peaks["bf16_tflops"],
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "tokens/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": Ke,
                    "api": "lsp_layer_step_host_async x K + lsp_host_copies_wait (pinned host x, dy in; y, dx out every step)"},
            "gpu_launches": int(launches), "per_step_ms": per_step, "roofline": roofline}

    if renv.is_main and renv.world_size == 1 and not args.no_cpu_baseline:
        tps, dt, sample = time_oracle(w, 3, 1) if args.cpu_baseline_sample else time_oracle_full(w)
        line["cpu_baseline"] = {"value": tps, "unit": "tokens/s", "cores": blas_threads(), "kind": "oracle", "sample": sample,
                                "s_per_step": dt, "nproc": host_cpu()[0], "cpu_model": host_cpu()[1]}
    ctx.close()
    replicas.finalize()
    if renv.is_main:
        print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg1", "cfg2", "cfg4"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--recast-weights", action="store_true",
                    help="convert the bf16 weights to fp16 operands inside every forward call instead of once before the loop")
    ap.add_argument("--cpu-baseline-sample", action="store_true",
                    help="time the oracle on the bounded sample (as --impl reference does) instead of one full-size step")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
