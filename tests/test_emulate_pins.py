"""Pins of oracle/emulate16.py (the oracle's 16-bit-operand emulation mode, used only to report the precision floor
beside a GPU error above the bar).  CPU only."""
import numpy as np

from oracle import emulate16 as E
from oracle import lspref as R


def _case(seed=3, B=2, S=48, H=64, nq=4, nkv=2, d=16, F=96):
    rng = np.random.default_rng(seed)
    cfg = R.LayerShape(B, S, H, nq, nkv, d, F, 1e-5, 10000.0)
    w = dict(wq=0.1 * rng.standard_normal((nq * d, H)), wk=0.1 * rng.standard_normal((nkv * d, H)),
             wv=0.1 * rng.standard_normal((nkv * d, H)), wo=0.1 * rng.standard_normal((H, nq * d)),
             w_gate=0.1 * rng.standard_normal((F, H)), w_up=0.1 * rng.standard_normal((F, H)),
             w_down=0.1 * rng.standard_normal((H, F)), g_attn=1 + 0.1 * rng.standard_normal(H), g_mlp=1 + 0.1 * rng.standard_normal(H))
    return cfg, w, rng.standard_normal((B * S, H)), rng.standard_normal((B * S, H))


def test_without_rounding_the_emulation_is_the_oracle():
    """fmt = "exact": every rounding site is the identity, so forward, backward (from the saved log-sum-exp and
    D = rowsum(dO * O) instead of the explicit softmax Jacobian) and the two-layer stack must reproduce lspref to
    round-off -- a wrong operand, transposition or missing term at any site of the emulation fails here."""
    cfg, w, x, dy = _case()
    ref = R.layer_fwd_bwd(x, dy, w, cfg)
    rnd = E.make_rounder("exact")
    y, c = E.layer_fwd(x, w, cfg, rnd)
    dx, g = E.layer_bwd(dy, w, cfg, c, rnd)
    np.testing.assert_allclose(y, ref["y"], rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(dx, ref["dx"], rtol=1e-9, atol=1e-11)
    for k, v in g.items():
        np.testing.assert_allclose(v, ref["d" + k], rtol=1e-9, atol=1e-10, err_msg=k)
    y2, d2, g2 = E.stack_fwd_bwd(x, dy, [w, w], cfg, fmt="exact")
    yr, dr, gr = R.stack_fwd_bwd(x, dy, [w, w], cfg)
    np.testing.assert_allclose(y2, yr, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(d2, dr, rtol=1e-9, atol=1e-11)
    for l in range(2):
        for k, v in g2[l].items():
            np.testing.assert_allclose(v, gr[l][k], rtol=1e-9, atol=1e-10, err_msg=f"{l}/{k}")


def test_rounding_sites_are_live_and_ordered():
    """With rounding on, every output differs from the oracle by a small, non-zero amount, and bf16 operands (8 mantissa
    bits) are several times worse than fp16 operands (11 bits) on every tensor."""
    cfg, w, x, dy = _case(seed=4)
    ref = R.layer_fwd_bwd(x, dy, w, cfg)
    errs = {}
    for fmt in ("f16", "bf16"):
        rnd = E.make_rounder(fmt)
        y, c = E.layer_fwd(x, w, cfg, rnd)
        dx, g = E.layer_bwd(dy, w, cfg, c, rnd, split_rows=0)
        out = dict(y=y, dx=dx, **{"d" + k: v for k, v in g.items()})
        errs[fmt] = {k: float(np.max(np.abs(v - ref[k])) / np.sqrt(np.mean(ref[k] ** 2))) for k, v in out.items()}
    for k in errs["f16"]:
        assert 0.0 < errs["f16"][k] < 2e-2, (k, errs["f16"][k])
        assert errs["bf16"][k] > 3.0 * errs["f16"][k], (k, errs)
    r16, rb = E.make_rounder("f16"), E.make_rounder("bf16")
    v = np.array([1.0 + 2.0 ** -11, 1.0 + 2.0 ** -10, 65520.0, 1e-8, 1.0 + 2.0 ** -8, 1.0 + 2.0 ** -9])
    np.testing.assert_array_equal(r16(v)[:2], [1.0, 1.0 + 2.0 ** -10])              # ties to even at 11 bits
    np.testing.assert_array_equal(rb(v)[4:], [1.0, 1.0])                            # 2^-8 is half an ulp of bf16: tie to even
