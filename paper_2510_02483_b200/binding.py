"""Thin ctypes binding over liblsp.so (include/lsp.h): argument marshalling only.

Every function has the name and argument order of its C entry point; tensors are torch CUDA tensors
(PyTorch is used for device memory and streams only) passed as raw device pointers.  There is no CPU
fallback: if liblsp.so is missing or a call fails, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "liblsp.so")

LSP_BF16, LSP_F32, LSP_F16 = 0, 1, 2
STATUS = {0: "LSP_OK", -1: "LSP_EINVAL", -2: "LSP_EUNSUPPORTED", -3: "LSP_ENOMEM", -4: "LSP_ECUDA", -5: "LSP_EALIGN"}
WEIGHT_FIELDS = ("wq", "wk", "wv", "wo", "g_attn", "w_gate", "w_up", "w_down", "g_mlp")
EXPORTS = ("lsp_create", "lsp_destroy", "lsp_saved_bytes", "lsp_workspace_bytes", "lsp_last_error",
           "lsp_attn_fwd", "lsp_attn_bwd", "lsp_mlp_fwd", "lsp_mlp_bwd", "lsp_layer_fwd", "lsp_layer_bwd",
           "lsp_sdpa_fwd", "lsp_sdpa_bwd", "lsp_embed_fwd", "lsp_gemm", "lsp_layer_step_host", "lsp_launch_count",
           "lsp_timing_enable", "lsp_timing_read", "lsp_adamw_step", "lsp_lr_cosine", "lsp_head_workspace_bytes",
           "lsp_head_fwd_bwd", "lsp_embed_bwd", "lsp_layer_step_host_async", "lsp_host_copies_wait", "lsp_set_packed_sequences", "lsp_layer_fwd_infer",
           "lsp_overflow_count", "lsp_weight_cache_bytes", "lsp_layer_prepare_weights", "lsp_weight_cache_offset",
           "lsp_grad_norm_static")


class LspError(RuntimeError):
    pass


class lsp_layer_desc(C.Structure):
    _fields_ = [("batch", C.c_int32), ("seq", C.c_int32), ("hidden", C.c_int32), ("n_q_heads", C.c_int32),
                ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32), ("ffn", C.c_int32), ("rms_eps", C.c_float),
                ("rope_base", C.c_double), ("rope_layout", C.c_int32), ("use_rope", C.c_int32),
                ("in_dtype", C.c_int32), ("wgrad_accumulate", C.c_int32), ("head_dim_logical", C.c_int32),
                ("residual_scale_set", C.c_int32), ("residual_scale", C.c_float)]


class lsp_layer_weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in WEIGHT_FIELDS] + [("f16_cache", C.c_void_p)]


class lsp_adamw_tensor(C.Structure):
    _fields_ = [("grad", C.c_void_p), ("master", C.c_void_p), ("m", C.c_void_p), ("v", C.c_void_p),
                ("weight_bf16", C.c_void_p), ("n", C.c_int64), ("decay", C.c_int32), ("weight_f16", C.c_void_p)]


class lsp_adamw_desc(C.Structure):
    _fields_ = [("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float),
                ("weight_decay", C.c_float), ("clip_norm", C.c_float), ("step", C.c_int32), ("grad_scale", C.c_float), ("phase", C.c_int32)]


class lsp_layer_wgrads(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in WEIGHT_FIELDS]


_lib = None


def lib():
    """Load liblsp.so (raises if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise LspError(f"{LIB_PATH} not found: build it with `python -m paper_2510_02483_b200.build`")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_int64
        L.lsp_create.argtypes = [C.POINTER(vp), C.POINTER(lsp_layer_desc), i32]
        L.lsp_destroy.argtypes = [vp]
        L.lsp_saved_bytes.argtypes = [vp]; L.lsp_saved_bytes.restype = C.c_size_t
        L.lsp_workspace_bytes.argtypes = [vp]; L.lsp_workspace_bytes.restype = C.c_size_t
        L.lsp_last_error.argtypes = [vp]; L.lsp_last_error.restype = C.c_char_p
        pw, pg = C.POINTER(lsp_layer_weights), C.POINTER(lsp_layer_wgrads)
        L.lsp_attn_fwd.argtypes = [vp, vp, pw, vp, vp, vp, vp]
        L.lsp_attn_bwd.argtypes = [vp, vp, vp, pw, vp, vp, pg, vp, vp]
        L.lsp_mlp_fwd.argtypes = [vp, vp, pw, vp, vp, vp, vp]
        L.lsp_mlp_bwd.argtypes = [vp, vp, vp, pw, vp, vp, pg, vp, vp]
        L.lsp_layer_fwd.argtypes = [vp, vp, pw, vp, vp, vp, vp]
        L.lsp_layer_fwd_infer.argtypes = [vp, vp, pw, vp, vp, vp, vp]
        L.lsp_layer_bwd.argtypes = [vp, vp, vp, pw, vp, vp, pg, vp, vp]
        L.lsp_sdpa_fwd.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
        L.lsp_sdpa_bwd.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.lsp_embed_fwd.argtypes = [vp, vp, vp, vp, vp]
        L.lsp_gemm.argtypes = [vp, i32, i32, i32, i32, vp, i64, i32, vp, i64, i32, vp, i64, vp]
        L.lsp_layer_step_host.argtypes = [vp, vp, vp, pw, vp, vp, pg, vp, vp, vp, vp, vp, vp, vp]
        L.lsp_layer_step_host_async.argtypes = [vp, vp, vp, pw, vp, vp, pg, vp, vp, vp, vp, vp, vp, vp]
        L.lsp_host_copies_wait.argtypes = [vp, vp]
        L.lsp_set_packed_sequences.argtypes = [vp, C.POINTER(C.c_int32), i32, vp]
        L.lsp_launch_count.argtypes = [vp]; L.lsp_launch_count.restype = C.c_longlong
        L.lsp_timing_enable.argtypes = [vp, i32]
        L.lsp_timing_read.argtypes = [vp, i32, C.POINTER(C.c_char_p), C.POINTER(C.c_float), C.POINTER(i32)]
        L.lsp_adamw_step.argtypes = [vp, i32, C.POINTER(lsp_adamw_tensor), C.POINTER(lsp_adamw_desc), vp, vp]
        L.lsp_lr_cosine.argtypes = [i32, C.c_double, C.c_double, i32, i32]
        L.lsp_lr_cosine.restype = C.c_double
        L.lsp_head_workspace_bytes.argtypes = [vp, i32]
        L.lsp_head_workspace_bytes.restype = C.c_size_t
        L.lsp_head_fwd_bwd.argtypes = [vp, vp, vp, vp, vp, i32, C.c_float, vp, vp, vp, vp, vp, vp, vp]
        L.lsp_embed_bwd.argtypes = [vp, vp, vp, i32, vp, vp]
        L.lsp_overflow_count.argtypes = [vp, C.POINTER(C.c_ulonglong), i32, vp]
        L.lsp_weight_cache_bytes.argtypes = [vp]
        L.lsp_weight_cache_bytes.restype = C.c_size_t
        L.lsp_layer_prepare_weights.argtypes = [vp, pw, vp, vp]
        L.lsp_weight_cache_offset.argtypes = [vp, i32]
        L.lsp_weight_cache_offset.restype = C.c_longlong
        L.lsp_grad_norm_static.argtypes = [i32, i32, C.POINTER(vp), C.POINTER(i64), C.c_float, C.c_float, vp, vp, C.c_char_p, C.c_size_t]
        for n in EXPORTS:
            if n not in ("lsp_saved_bytes", "lsp_workspace_bytes", "lsp_last_error", "lsp_launch_count", "lsp_lr_cosine",
                         "lsp_head_workspace_bytes", "lsp_weight_cache_bytes", "lsp_weight_cache_offset"):
                getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _pack(struct_t, tensors: dict):
    """tensors: {field: torch tensor}; weights may carry "f16_cache" (a buffer filled by lsp_layer_prepare_weights)."""
    s = struct_t()
    for n in WEIGHT_FIELDS:
        t = tensors.get(n)
        setattr(s, n, None if t is None else t.data_ptr())
    if struct_t is lsp_layer_weights:
        t = tensors.get("f16_cache")
        s.f16_cache = None if t is None else t.data_ptr()
    return s


class Ctx:
    """Owns one lsp_ctx (a layer shape on a device)."""

    def __init__(self, *, batch, seq, hidden, n_q_heads, n_kv_heads, head_dim, ffn, rms_eps=1e-5, rope_base=10000.0,
                 use_rope=True, in_dtype=LSP_BF16, device=0, rope_layout=0, wgrad_accumulate=False, head_dim_logical=0, residual_scale=None):
        self.desc = lsp_layer_desc(batch, seq, hidden, n_q_heads, n_kv_heads, head_dim, ffn, rms_eps, rope_base, rope_layout,
                                   1 if use_rope else 0, in_dtype, 1 if wgrad_accumulate else 0, head_dim_logical,
                                   0 if residual_scale is None else 1, 1.0 if residual_scale is None else float(residual_scale))
        self.handle = C.c_void_p()
        st = lib().lsp_create(C.byref(self.handle), C.byref(self.desc), device)
        if st != 0:
            self.handle = None
            raise LspError(f"lsp_create failed: {STATUS.get(st, st)}")

    def close(self):
        if self.handle:
            lib().lsp_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def check(self, st):
        if st != 0:
            raise LspError(f"{STATUS.get(st, st)}: {lib().lsp_last_error(self.handle).decode()}")

    @property
    def saved_bytes(self):
        return lib().lsp_saved_bytes(self.handle)

    @property
    def workspace_bytes(self):
        return lib().lsp_workspace_bytes(self.handle)

    @property
    def weight_cache_bytes(self):
        return lib().lsp_weight_cache_bytes(self.handle)


def lsp_attn_fwd(ctx, x, weights, a_out, saved, ws, stream=None):
    w = _pack(lsp_layer_weights, weights)
    ctx.check(lib().lsp_attn_fwd(ctx.handle, _ptr(x), C.byref(w), _ptr(a_out), _ptr(saved), _ptr(ws), _stream(stream)))


def lsp_attn_bwd(ctx, x, da, weights, saved, dx, grads, ws, stream=None):
    w, g = _pack(lsp_layer_weights, weights), _pack(lsp_layer_wgrads, grads)
    ctx.check(lib().lsp_attn_bwd(ctx.handle, _ptr(x), _ptr(da), C.byref(w), _ptr(saved), _ptr(dx), C.byref(g), _ptr(ws),
                                 _stream(stream)))


def lsp_mlp_fwd(ctx, a, weights, y_out, saved, ws, stream=None):
    w = _pack(lsp_layer_weights, weights)
    ctx.check(lib().lsp_mlp_fwd(ctx.handle, _ptr(a), C.byref(w), _ptr(y_out), _ptr(saved), _ptr(ws), _stream(stream)))


def lsp_mlp_bwd(ctx, a, dy, weights, saved, da, grads, ws, stream=None):
    w, g = _pack(lsp_layer_weights, weights), _pack(lsp_layer_wgrads, grads)
    ctx.check(lib().lsp_mlp_bwd(ctx.handle, _ptr(a), _ptr(dy), C.byref(w), _ptr(saved), _ptr(da), C.byref(g), _ptr(ws),
                                _stream(stream)))


def lsp_layer_fwd_infer(ctx, x, weights, y_out, scratch, ws, stream=None):
    w = _pack(lsp_layer_weights, weights)
    ctx.check(lib().lsp_layer_fwd_infer(ctx.handle, _ptr(x), C.byref(w), _ptr(y_out), _ptr(scratch), _ptr(ws), _stream(stream)))


def lsp_layer_fwd(ctx, x, weights, y_out, saved, ws, stream=None):
    w = _pack(lsp_layer_weights, weights)
    ctx.check(lib().lsp_layer_fwd(ctx.handle, _ptr(x), C.byref(w), _ptr(y_out), _ptr(saved), _ptr(ws), _stream(stream)))


def lsp_layer_bwd(ctx, x, dy, weights, saved, dx, grads, ws, stream=None):
    w, g = _pack(lsp_layer_weights, weights), _pack(lsp_layer_wgrads, grads)
    ctx.check(lib().lsp_layer_bwd(ctx.handle, _ptr(x), _ptr(dy), C.byref(w), _ptr(saved), _ptr(dx), C.byref(g), _ptr(ws),
                                  _stream(stream)))


def lsp_sdpa_fwd(ctx, q, k, v, o, lse, ws, stream=None):
    ctx.check(lib().lsp_sdpa_fwd(ctx.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(o), _ptr(lse), _ptr(ws), _stream(stream)))


def lsp_sdpa_bwd(ctx, q, k, v, o, lse, d_o, dq, dk, dv, ws, stream=None):
    ctx.check(lib().lsp_sdpa_bwd(ctx.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(o), _ptr(lse), _ptr(d_o), _ptr(dq), _ptr(dk),
                                 _ptr(dv), _ptr(ws), _stream(stream)))


def lsp_embed_fwd(ctx, ids, table, x0, stream=None):
    ctx.check(lib().lsp_embed_fwd(ctx.handle, _ptr(ids), _ptr(table), _ptr(x0), _stream(stream)))


def lsp_gemm(ctx, op, M, N, K, A, lda, a_dtype, B, ldb, b_dtype, Cout, ldc, stream=None):
    ctx.check(lib().lsp_gemm(ctx.handle, op, M, N, K, _ptr(A), lda, a_dtype, _ptr(B), ldb, b_dtype, _ptr(Cout), ldc,
                             _stream(stream)))


def lsp_layer_step_host(ctx, x_host, dy_host, weights, y_host, dx_host, grads, x_dev, dy_dev, y_dev, dx_dev, saved, ws,
                        stream=None):
    w, g = _pack(lsp_layer_weights, weights), _pack(lsp_layer_wgrads, grads)
    ctx.check(lib().lsp_layer_step_host(ctx.handle, _ptr(x_host), _ptr(dy_host), C.byref(w), _ptr(y_host), _ptr(dx_host),
                                        C.byref(g), _ptr(x_dev), _ptr(dy_dev), _ptr(y_dev), _ptr(dx_dev), _ptr(saved),
                                        _ptr(ws), _stream(stream)))


def lsp_layer_step_host_async(ctx, x_host, dy_host, weights, y_host, dx_host, grads, x_dev, dy_dev, y_dev, dx_dev, saved, ws,
                              stream=None):
    w, g = _pack(lsp_layer_weights, weights), _pack(lsp_layer_wgrads, grads)
    ctx.check(lib().lsp_layer_step_host_async(ctx.handle, _ptr(x_host), _ptr(dy_host), C.byref(w), _ptr(y_host), _ptr(dx_host),
                                              C.byref(g), _ptr(x_dev), _ptr(dy_dev), _ptr(y_dev), _ptr(dx_dev), _ptr(saved),
                                              _ptr(ws), _stream(stream)))


def lsp_set_packed_sequences(ctx, cu_seqlens, stream=None):
    """cu_seqlens: host sequence of n_seqs + 1 ints (0 ... total tokens); empty / None switches packing off."""
    n = 0 if not cu_seqlens else len(cu_seqlens) - 1
    arr = (C.c_int32 * (n + 1))(*([0] if n == 0 else [int(v) for v in cu_seqlens]))
    ctx.check(lib().lsp_set_packed_sequences(ctx.handle, arr, n, _stream(stream)))


def lsp_layer_prepare_weights(ctx, weights, cache, stream=None):
    w = _pack(lsp_layer_weights, weights)
    ctx.check(lib().lsp_layer_prepare_weights(ctx.handle, C.byref(w), _ptr(cache), _stream(stream)))


def lsp_weight_cache_bytes(ctx) -> int:
    return int(lib().lsp_weight_cache_bytes(ctx.handle))


def lsp_weight_cache_offset(ctx, which: int) -> int:
    return int(lib().lsp_weight_cache_offset(ctx.handle, which))


def lsp_overflow_count(ctx, reset=False, stream=None) -> int:
    n = C.c_ulonglong(0)
    ctx.check(lib().lsp_overflow_count(ctx.handle, C.byref(n), 1 if reset else 0, _stream(stream)))
    return int(n.value)


def lsp_host_copies_wait(ctx, stream=None):
    ctx.check(lib().lsp_host_copies_wait(ctx.handle, _stream(stream)))


def lsp_adamw_step(ctx, tensors, *, lr, step, gnorm_out, beta1=0.90, beta2=0.95, eps=1e-8, weight_decay=0.01, clip_norm=1.0,
                   grad_scale=1.0, phase=0, stream=None):
    """tensors: list of dicts {grad, master, m, v, weight (bf16 or None), decay (bool), weight_f16 (fp16 view or None)} of
    torch CUDA tensors."""
    arr = (lsp_adamw_tensor * len(tensors))()
    for i, t in enumerate(tensors):
        w, w16 = t.get("weight"), t.get("weight_f16")
        arr[i] = lsp_adamw_tensor(t["grad"].data_ptr(), t["master"].data_ptr(), t["m"].data_ptr(), t["v"].data_ptr(),
                                  None if w is None else w.data_ptr(), t["master"].numel(), 1 if t.get("decay", True) else 0,
                                  None if w16 is None else w16.data_ptr())
    d = lsp_adamw_desc(lr, beta1, beta2, eps, weight_decay, clip_norm, step, grad_scale, phase)
    ctx.check(lib().lsp_adamw_step(ctx.handle, len(tensors), arr, C.byref(d), _ptr(gnorm_out), _stream(stream)))


NORM_STATIC_MAX_TENSORS = 256            # LSP_NORM_STATIC_MAX_TENSORS of include/lsp.h


def lsp_grad_norm_static(grads, gnorm_out, *, clip_norm=1.0, grad_scale=1.0, stream=None):
    """Allocation-free global gradient norm (include/lsp.h): grads = list of fp32 torch CUDA tensors on one device,
    gnorm_out = fp32 CUDA tensor of 2 elements.  Needs no Ctx; the scratch is a static device array of the library."""
    k = len(grads)
    ptrs = (C.c_void_p * max(k, 1))(*[g.data_ptr() for g in grads])
    ns = (C.c_int64 * max(k, 1))(*[g.numel() for g in grads])
    err = C.create_string_buffer(512)
    dev = gnorm_out.device.index if gnorm_out.device.index is not None else 0
    st = lib().lsp_grad_norm_static(dev, k, ptrs, ns, C.c_float(clip_norm), C.c_float(grad_scale), _ptr(gnorm_out), _stream(stream), err, len(err))
    if st != 0:
        raise LspError(f"{STATUS.get(st, st)}: {err.value.decode(errors='replace')}")


def lsp_lr_cosine(step: int, lr_max: float = 1.2e-3, lr_min: float = 1.0e-5, warmup: int = 2000, total: int = 100000) -> float:
    return float(lib().lsp_lr_cosine(step, lr_max, lr_min, warmup, total))


def lsp_head_workspace_bytes(ctx, vocab: int) -> int:
    return int(lib().lsp_head_workspace_bytes(ctx.handle, vocab))


def lsp_head_fwd_bwd(ctx, x, g_final, w_head, targets, vocab, loss, lse, dx, dg_final, dw_head, ws, stream=None, grad_scale=1.0):
    ctx.check(lib().lsp_head_fwd_bwd(ctx.handle, _ptr(x), _ptr(g_final), _ptr(w_head), _ptr(targets), vocab, grad_scale, _ptr(loss), _ptr(lse),
                                     _ptr(dx), _ptr(dg_final), _ptr(dw_head), _ptr(ws), _stream(stream)))


def lsp_embed_bwd(ctx, ids, dx0, vocab, d_table, stream=None):
    ctx.check(lib().lsp_embed_bwd(ctx.handle, _ptr(ids), _ptr(dx0), vocab, _ptr(d_table), _stream(stream)))


def lsp_launch_count(ctx) -> int:
    return int(lib().lsp_launch_count(ctx.handle))


def lsp_timing_enable(ctx, max_records: int):
    ctx.check(lib().lsp_timing_enable(ctx.handle, max_records))


def lsp_timing_read(ctx) -> dict:
    """{stage name: (total_ms, records)} for the stages recorded since the last read."""
    n = 64
    names, ms, cnt = (C.c_char_p * n)(), (C.c_float * n)(), (C.c_int * n)()
    k = lib().lsp_timing_read(ctx.handle, n, names, ms, cnt)
    if k < 0:
        raise LspError("lsp_timing_read failed")
    return {names[i].decode(): (float(ms[i]), int(cnt[i])) for i in range(k) if cnt[i] > 0}
