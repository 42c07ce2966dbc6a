"""lsp_grad_norm_static: the allocation-free gradient-norm entry point (include/lsp.h) against the existing path.

Collected LAST on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide another test.

The existing path is the norm / clipping pass of lsp_adamw_step (phase 0), whose partial sums live in a buffer the
context allocated; the new entry point runs the same kernels with the partial sums in a static device array of the
library and needs no context.  Both reduce in the same fixed order, so gnorm_out must agree BIT FOR BIT (tighter than
the 1e-6 relative bar tests/test_gpu_parity.py::test_adamw_step_vs_oracle holds the norm to, which is also asserted
against a float64 sum here so that the test says something when run alone).  Two calls in a row on different gradient
sets (the second smaller: the array still holds the first call's partial sums, none of which may be read), a call
beyond the stated maximum (rejected with a message, nothing launched), and the caller's memory footprint (no device
allocation during the calls)."""
import numpy as np
import pytest


def _reference(ctx, B, grads, clip_norm, grad_scale, dev):
    """gnorm_out of lsp_adamw_step phase 0 on the same gradients (throw-away optimizer state)."""
    import torch
    gn = torch.zeros(2, dtype=torch.float32, device=dev)
    tensors = [dict(grad=g, master=torch.zeros_like(g), m=torch.zeros_like(g), v=torch.zeros_like(g), weight=None, decay=False)
               for g in grads]
    B.lsp_adamw_step(ctx, tensors, lr=1e-3, step=1, gnorm_out=gn, clip_norm=clip_norm, grad_scale=grad_scale)
    torch.cuda.synchronize()
    return gn


@pytest.mark.gpu
def test_grad_norm_static_matches_adamw_norm_pass_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_2510_02483_b200 import binding as B
    from paper_2510_02483_b200 import harness, synth
    B.lib()
    dev = torch.device("cuda", torch.cuda.current_device())
    gen = torch.Generator(device="cpu").manual_seed(251002483)
    # call 1: 37 tensors (three kernel groups of 16), ragged sizes, one large enough for the grid-stride loop
    # (> 148 * 8 blocks of 256 float4); call 2: 3 small tensors, stored scaled by 64, norm below the clip threshold
    shapes1 = [(3072, 1024), (1000, 64), (512,), (36, 100), (4,)] + [(128 + 4 * i, 12) for i in range(32)]
    shapes2 = [(260, 64), (8,), (52, 100)]
    sets = [([(torch.randn(s, generator=gen) * 0.05).to(dev) for s in shapes1], 1.0, 1.0),
            ([(torch.randn(s, generator=gen) * 1e-4 * 64.0).to(dev) for s in shapes2], 0.5, 64.0)]
    ctx = harness.make_ctx(synth.CFG1_TINY)
    want = [_reference(ctx, B, g, clip, gs, dev) for g, clip, gs in sets]
    ctx.close()                                   # the new entry point needs no context
    out = [torch.full((2,), -1.0, dtype=torch.float32, device=dev) for _ in sets]
    B.lsp_grad_norm_static(sets[0][0], out[0], clip_norm=sets[0][1], grad_scale=sets[0][2])      # set-up call
    torch.cuda.synchronize()
    exact = [float(np.sqrt(sum(float((x.double() ** 2).sum()) for x in g))) / gs for g, _, gs in sets]
    mem0 = None
    for it in range(3):                           # rounds of two calls in a row, no sync in between
        for o in out:
            o.fill_(-1.0)
        for (g, clip, gs), o in zip(sets, out):
            B.lsp_grad_norm_static(g, o, clip_norm=clip, grad_scale=gs)
        torch.cuda.synchronize()
        for (g, clip, gs), o, w, ex in zip(sets, out, want, exact):
            assert torch.equal(o.view(torch.int32), w.view(torch.int32)), (o.tolist(), w.tolist())
            n, c = o.tolist()
            assert abs(n - ex) <= 1e-6 * ex
            assert abs(c * gs - min(1.0, clip / (ex + 1e-6))) <= 2e-6
        if it == 0:                               # after one round: torch's own caching allocator has what it needs
            mem0 = torch.cuda.mem_get_info()[0]
    assert torch.cuda.mem_get_info()[0] >= mem0   # the calls took no device memory
    # a non-finite gradient: {non-finite norm, 0}, as on the existing path
    sets[1][0][1][3] = float("inf")
    B.lsp_grad_norm_static(sets[1][0], out[1], clip_norm=0.5, grad_scale=64.0)
    torch.cuda.synchronize()
    n, c = out[1].tolist()
    assert not np.isfinite(n) and c == 0.0
    # beyond the maximum: rejected with a message, the output untouched
    out[0].fill_(-1.0)
    many = [sets[0][0][2]] * (B.NORM_STATIC_MAX_TENSORS + 1)
    with pytest.raises(B.LspError, match="LSP_EINVAL.*exceed the maximum of 256"):
        B.lsp_grad_norm_static(many, out[0])
    with pytest.raises(B.LspError, match="LSP_EINVAL"):
        B.lsp_grad_norm_static([], out[0])
    with pytest.raises(B.LspError, match="n % 4"):
        B.lsp_grad_norm_static([torch.zeros(6, dtype=torch.float32, device=dev)], out[0])
    torch.cuda.synchronize()
    assert out[0].tolist() == [-1.0, -1.0]
    # exactly at the maximum: accepted
    B.lsp_grad_norm_static(many[:B.NORM_STATIC_MAX_TENSORS], out[0])
    torch.cuda.synchronize()
    exact = float(np.sqrt(B.NORM_STATIC_MAX_TENSORS * float((sets[0][0][2].double() ** 2).sum())))
    assert abs(out[0].tolist()[0] - exact) <= 1e-6 * exact


def test_grad_norm_static_rejects_sizes_beyond_the_maximum_without_a_gpu():
    """The size checks come before any CUDA call: a request beyond LSP_NORM_STATIC_MAX_TENSORS (or a malformed one) is a
    status plus a message in the caller's buffer, on a machine without a GPU too."""
    import ctypes as C
    from paper_2510_02483_b200 import binding as B
    L = B.lib()
    err = C.create_string_buffer(256)
    k = B.NORM_STATIC_MAX_TENSORS + 1
    ptrs = (C.c_void_p * k)(*([256] * k))                  # never dereferenced: the call is rejected first
    ns = (C.c_int64 * k)(*([8] * k))
    out = C.c_void_p(512)
    assert L.lsp_grad_norm_static(0, k, ptrs, ns, 1.0, 1.0, out, None, err, len(err)) == -1
    assert b"exceed the maximum of 256" in err.value
    assert L.lsp_grad_norm_static(0, 0, ptrs, ns, 1.0, 1.0, out, None, err, len(err)) == -1 and b"ntensors" in err.value
    ns[1] = 6
    assert L.lsp_grad_norm_static(0, 2, ptrs, ns, 1.0, 1.0, out, None, err, len(err)) == -1 and b"tensor 1" in err.value
    ns[1] = 8
    ptrs[1] = 264
    assert L.lsp_grad_norm_static(0, 2, ptrs, ns, 1.0, 1.0, out, None, err, len(err)) == -5 and b"aligned" in err.value
    assert L.lsp_grad_norm_static(0, 2, ptrs, ns, 0.0, 1.0, out, None, None, 0) == -1      # err may be NULL
