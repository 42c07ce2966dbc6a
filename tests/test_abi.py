"""CPU-side checks of the boundary: liblsp.so builds for sm_100a, loads, and exports every entry point that
include/lsp.h declares (no compute calls: there is no GPU here), and the binding mirrors the same names."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2510_02483_b200 import build
    return build.build()           # no-op when the in-tree .so is up to date


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "lsp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lsp_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_north_star_calls():
    names = declared_symbols()
    for n in ("lsp_attn_fwd", "lsp_attn_bwd", "lsp_mlp_fwd", "lsp_mlp_bwd", "lsp_layer_fwd", "lsp_layer_bwd"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for n in declared_symbols():
        assert hasattr(lib, n), f"liblsp.so does not export {n}"


def test_binding_mirrors_header(libpath):
    from paper_2510_02483_b200 import binding
    binding.lib()
    assert sorted(binding.EXPORTS) == declared_symbols()
    for n in declared_symbols():
        if n not in ("lsp_create", "lsp_destroy", "lsp_saved_bytes", "lsp_workspace_bytes", "lsp_last_error"):
            assert callable(getattr(binding, n)), n


def test_null_arguments_are_rejected_without_a_gpu(libpath):
    lib = ctypes.CDLL(libpath)
    lib.lsp_create.restype = ctypes.c_int
    assert lib.lsp_create(None, None, 0) == -1          # LSP_EINVAL
    lib.lsp_layer_fwd.restype = ctypes.c_int
    assert lib.lsp_layer_fwd(None, None, None, None, None, None, None) == -1


def test_create_rejects_bad_shapes_without_a_gpu(libpath):
    """lsp_create checks the descriptor before it touches the device: empty and unsupported shapes come back as a
    status, never as a crash or a silent fallback (include/lsp.h, error behaviour)."""
    from paper_2510_02483_b200 import binding as B
    B.lib()
    ok = dict(batch=1, seq=128, hidden=256, n_q_heads=4, n_kv_heads=2, head_dim=64, ffn=688)
    cases = [(dict(batch=0), "LSP_EINVAL"), (dict(seq=0), "LSP_EINVAL"), (dict(n_kv_heads=3), "LSP_EINVAL"),
             (dict(head_dim=96), "LSP_EUNSUPPORTED"), (dict(hidden=260), "LSP_EUNSUPPORTED"), (dict(ffn=690), "LSP_EUNSUPPORTED"),
             (dict(hidden=16384), "LSP_EUNSUPPORTED"), (dict(rope_layout=2), "LSP_EUNSUPPORTED"),
             (dict(head_dim_logical=51), "LSP_EUNSUPPORTED"), (dict(head_dim_logical=80), "LSP_EUNSUPPORTED"),
             (dict(head_dim_logical=52, rope_layout=1), "LSP_EUNSUPPORTED"), (dict(rope_base=0.0), "LSP_EINVAL"),
             (dict(in_dtype=7), "LSP_EINVAL"), (dict(batch=1 << 20, seq=1 << 12), "LSP_EUNSUPPORTED")]
    for kw, status in cases:
        with pytest.raises(B.LspError, match=status):
            B.Ctx(**dict(ok, **kw))


def test_sass_is_blackwell_native(libpath):
    """The GEMM kernels must contain tcgen05 MMA (UTC*MMA), TMEM loads (LDTM) and TMA loads (UTMALDG)."""
    import subprocess
    cuobjdump = "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", libpath], capture_output=True, text=True).stdout
    assert re.search(r"UTC[A-Z]*MMA", sass) and "LDTM" in sass and "UTMALDG" in sass
    assert "UTMASTG" in sass and "UTMAREDG" in sass          # TMA tensor stores and reduce-add stores (epilogues, wgrad accumulation)


def test_lr_cosine_host_helper_matches_oracle(libpath):
    """lsp_lr_cosine is host-only arithmetic (PAPER.md:77 schedule, reading O-3): identical to the oracle's schedule."""
    from oracle import adamw_ref as A
    from paper_2510_02483_b200 import binding
    for total in (5000, 100000):
        for step in (1, 2, 999, 2000, 2001, 2500, total // 2, total - 1, total, total + 7):
            assert binding.lsp_lr_cosine(step, 1.2e-3, 1.0e-5, 2000, total) == pytest.approx(A.lr_cosine(step, total=total), rel=1e-14)
