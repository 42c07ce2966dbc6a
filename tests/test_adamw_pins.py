"""Pins of the fp64 AdamW oracle (oracle/adamw_ref.py) against what the paper and the mathematics fix: the Table-2
hyper-parameters, closed forms of the first step, invariants of clipping and of the schedule, and
torch.optim.AdamW / clip_grad_norm_ in float64 as an independent library second opinion.  CPU only."""
import math

import numpy as np
import pytest

from oracle import adamw_ref as A


def _rand(seed, shapes, scale=1.0):
    rng = np.random.default_rng(seed)
    return [rng.standard_normal(s) * scale for s in shapes]


SHAPES = [(7, 5), (11,), (3, 4)]


def test_table2_hyperparameters():
    """PAPER.md:73,77 and Table 2."""
    assert (A.BETA1, A.BETA2, A.WEIGHT_DECAY, A.CLIP_NORM) == (0.90, 0.95, 0.01, 1.0)
    assert (A.LR_MAX, A.LR_MIN, A.WARMUP) == (1.2e-3, 1.0e-5, 2000)


def test_schedule_closed_forms():
    total = 10000
    assert A.lr_cosine(1000, total=total) == pytest.approx(0.6e-3, rel=1e-15)           # half-way through the warm-up
    assert A.lr_cosine(2000, total=total) == pytest.approx(1.2e-3, rel=1e-15)           # end of the warm-up = maximum
    assert A.lr_cosine(total, total=total) == pytest.approx(1.0e-5, rel=1e-15)          # end of the cosine = minimum
    assert A.lr_cosine(total + 500, total=total) == 1.0e-5
    assert A.lr_cosine(6000, total=total) == pytest.approx(0.5 * (1.2e-3 + 1.0e-5), rel=1e-12)   # midpoint: cos(pi/2) = 0
    lrs = [A.lr_cosine(t, total=total) for t in range(1, total + 1)]
    assert all(b > a for a, b in zip(lrs[:1999], lrs[1:2000]))                          # strictly increasing warm-up
    assert all(b < a for a, b in zip(lrs[1999:-1], lrs[2000:]))                         # strictly decreasing afterwards
    # symmetry of the cosine about its midpoint
    assert A.lr_cosine(3000, total=total) + A.lr_cosine(9000, total=total) == pytest.approx(1.2e-3 + 1.0e-5, rel=1e-12)


def test_global_norm_and_clipping_invariants():
    g = _rand(1, SHAPES, 3.0)
    flat = np.concatenate([x.reshape(-1) for x in g])
    assert A.global_grad_norm(g) == pytest.approx(float(np.linalg.norm(flat)), rel=1e-14)
    n = A.global_grad_norm(g)
    c = A.clip_coefficient(n)
    assert c < 1.0 and A.global_grad_norm([x * c for x in g]) <= 1.0                    # clipped norm <= threshold
    small = [x * (0.5 / n) for x in g]
    assert A.clip_coefficient(A.global_grad_norm(small)) == 1.0                          # below the threshold: untouched
    # clipping makes the step invariant to a positive rescaling of an over-threshold gradient
    p = _rand(2, SHAPES, 0.02); z = [np.zeros(s) for s in SHAPES]
    a, _, _, _ = A.adamw_step(p, g, z, z, [1, 0, 1], 1, 1e-3)
    b, _, _, _ = A.adamw_step(p, [x * 7.0 for x in g], z, z, [1, 0, 1], 1, 1e-3)
    for x, y in zip(a, b):
        np.testing.assert_allclose(x, y, rtol=0, atol=1e-9)


def test_first_step_closed_form():
    """From zero moments: m_hat = g, v_hat = g^2, so the step is lr (g / (|g| + eps) + wd p) -- sign(g) up to eps."""
    p = _rand(3, SHAPES, 0.02); g = _rand(4, SHAPES, 1e-3)          # norm far below the clip threshold
    z = [np.zeros(s) for s in SHAPES]
    lr = 1.2e-3
    out, m, v, _ = A.adamw_step(p, g, z, z, [1, 1, 0], 1, lr)
    for i, dec in enumerate([1, 1, 0]):
        expect = p[i] - lr * (g[i] / (np.abs(g[i]) + A.EPS) + (A.WEIGHT_DECAY if dec else 0.0) * p[i])
        np.testing.assert_allclose(out[i], expect, rtol=1e-12, atol=0)
        np.testing.assert_allclose(m[i], 0.1 * g[i], rtol=1e-13)
        np.testing.assert_allclose(v[i], 0.05 * g[i] ** 2, rtol=1e-12)


def test_zero_gradient_only_decays():
    p = _rand(5, SHAPES, 0.02); z = [np.zeros(s) for s in SHAPES]
    out, m, v, n = A.adamw_step(p, z, z, z, [1, 0, 1], 3, 1e-3)
    assert n == 0.0
    np.testing.assert_allclose(out[0], p[0] * (1 - 1e-3 * 0.01), rtol=1e-15)
    np.testing.assert_array_equal(out[1], p[1])                      # gains: no decay (reading O-4)
    assert not np.any(m[0]) and not np.any(v[0])


def test_against_torch_adamw_float64():
    """Five steps against torch.optim.AdamW + clip_grad_norm_ (float64): same decoupled decay, bias correction, eps
    placement and global-norm clipping."""
    import torch
    shapes = SHAPES
    p0 = _rand(6, shapes, 0.02)
    tp = [torch.tensor(x, dtype=torch.float64, requires_grad=True) for x in p0]
    opt = torch.optim.AdamW([{"params": [tp[0], tp[2]], "weight_decay": 0.01}, {"params": [tp[1]], "weight_decay": 0.0}],
                            lr=1e-3, betas=(0.90, 0.95), eps=1e-8)
    p = [x.copy() for x in p0]; m = [np.zeros(s) for s in shapes]; v = [np.zeros(s) for s in shapes]
    for step in range(1, 6):
        g = _rand(100 + step, shapes, 2.0 if step % 2 else 0.05)     # alternately above and below the clip threshold
        lr = A.lr_cosine(step * 700, total=5000)
        for group in opt.param_groups:
            group["lr"] = lr
        for t, gi in zip(tp, g):
            t.grad = torch.tensor(gi, dtype=torch.float64)
        tn = torch.nn.utils.clip_grad_norm_(tp, 1.0)
        opt.step()
        p, m, v, n = A.adamw_step(p, g, m, v, [1, 0, 1], step, lr)
        assert n == pytest.approx(float(tn), rel=1e-12)
        for a, b in zip(p, tp):
            np.testing.assert_allclose(a, b.detach().numpy(), rtol=1e-11, atol=1e-15)


def test_bf16_rounding():
    x = np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 2.0 ** -7, 1.0 + 3 * 2.0 ** -8, -0.02, 3.1415926535])
    r = A.bf16_rne(x)
    assert r[0] == 1.0 and r[1] == 1.0                    # tie -> even (1.0 has an even mantissa)
    assert r[2] == 1.0 + 2.0 ** -7 and r[3] == 1.0 + 2.0 ** -6   # tie at 1 + 3/256 -> even neighbour 1 + 4/256
    assert np.all(np.abs(r - x) <= np.abs(x) * 2.0 ** -8)
    assert math.isclose(r[5], 3.140625)
