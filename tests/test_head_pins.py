"""Pins of the fp64 head/loss oracle (oracle/head_ref.py): closed forms, invariants, central finite differences and
torch float64 (rms_norm + linear + cross_entropy under autograd) as an independent library second opinion.  CPU only."""
import math

import numpy as np
import pytest

from oracle import head_ref as Hd

EPS = 1e-5


def _case(seed, T=12, H=16, V=37):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((T, H)), 1.0 + 0.1 * rng.standard_normal(H), 0.3 * rng.standard_normal((V, H)),
            rng.integers(0, V, size=T))


def test_uniform_logits_closed_form():
    """W_head = 0: every logit is 0, so loss = ln V, lse = ln V, dz = (1/V - onehot)/T and dx = dg = 0."""
    x, g, w, y = _case(1)
    V, T = w.shape[0], x.shape[0]
    out = Hd.head_loss_fwd_bwd(x, g, np.zeros_like(w), y, EPS)
    assert out["loss"] == pytest.approx(math.log(V), rel=1e-14)
    np.testing.assert_allclose(out["lse"], math.log(V), rtol=1e-14)
    assert not np.any(out["dx"]) and not np.any(out["dg_final"])
    xn = x / np.sqrt(np.mean(x * x, axis=1) + EPS)[:, None] * g
    onehot = np.zeros((T, V)); onehot[np.arange(T), y] = 1.0
    np.testing.assert_allclose(out["dw_head"], ((1.0 / V - onehot) / T).T @ xn, rtol=1e-12, atol=1e-15)


def test_invariants():
    x, g, w, y = _case(2)
    out = Hd.head_loss_fwd_bwd(x, g, w, y, EPS)
    # adding a constant to every logit of a token (a rank-one change of W along xn's null direction is awkward; instead:
    # shifting W_head by the same row vector c for all classes adds c.xn_t to every logit of token t) leaves the loss alone
    c = np.random.default_rng(3).standard_normal(w.shape[1])
    out2 = Hd.head_loss_fwd_bwd(x, g, w + c[None, :], y, EPS)
    assert out2["loss"] == pytest.approx(out["loss"], rel=1e-12)
    np.testing.assert_allclose(out2["dx"], out["dx"], rtol=1e-9, atol=1e-13)
    # the class gradients of every token sum to zero: sum_v dW_head[v,:] = sum_t (sum_v dz_tv) xn_t = 0
    np.testing.assert_allclose(np.sum(out["dw_head"], axis=0), 0.0, atol=1e-14)
    # one token, class 0 with logit alpha and V - 1 classes with logit 0: loss = log(1 + (V - 1) exp(-alpha)) exactly
    xn = x / np.sqrt(np.mean(x * x, axis=1) + EPS)[:, None] * g
    alpha, V1 = 3.0, 5
    w1 = np.vstack([alpha * xn[0] / np.dot(xn[0], xn[0]), np.zeros((V1 - 1, x.shape[1]))])
    o1 = Hd.head_loss_fwd_bwd(x[:1], g, w1, np.zeros(1, dtype=np.int64), EPS)
    assert o1["loss"] == pytest.approx(math.log(1.0 + (V1 - 1) * math.exp(-alpha)), rel=1e-13)


def test_finite_differences():
    x, g, w, y = _case(4, T=6, H=10, V=13)
    out = Hd.head_loss_fwd_bwd(x, g, w, y, EPS)
    rng = np.random.default_rng(5)
    h = 1e-6
    for name, arr, grad in (("x", x, out["dx"]), ("g", g, out["dg_final"]), ("w", w, out["dw_head"])):
        d = rng.standard_normal(arr.shape); d /= np.linalg.norm(d)
        args_p = dict(x=x, g=g, w=w); args_m = dict(x=x, g=g, w=w)
        args_p[name] = arr + h * d; args_m[name] = arr - h * d
        lp = Hd.head_loss_fwd_bwd(args_p["x"], args_p["g"], args_p["w"], y, EPS)["loss"]
        lm = Hd.head_loss_fwd_bwd(args_m["x"], args_m["g"], args_m["w"], y, EPS)["loss"]
        assert (lp - lm) / (2 * h) == pytest.approx(float(np.sum(grad * d)), rel=1e-6, abs=1e-9), name


def test_against_torch_float64():
    import torch
    import torch.nn.functional as F
    x, g, w, y = _case(6, T=20, H=24, V=50)
    out = Hd.head_loss_fwd_bwd(x, g, w, y, EPS)
    tx = torch.tensor(x, requires_grad=True); tg = torch.tensor(g, requires_grad=True); tw = torch.tensor(w, requires_grad=True)
    z = F.linear(F.rms_norm(tx, (x.shape[1],), tg, EPS), tw)
    loss = F.cross_entropy(z, torch.tensor(y))
    loss.backward()
    assert out["loss"] == pytest.approx(float(loss.detach()), rel=1e-13)
    np.testing.assert_allclose(out["lse"], torch.logsumexp(z, dim=1).detach().numpy(), rtol=1e-13)
    np.testing.assert_allclose(out["dx"], tx.grad.numpy(), rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(out["dg_final"], tg.grad.numpy(), rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(out["dw_head"], tw.grad.numpy(), rtol=1e-10, atol=1e-15)


def test_ignored_targets():
    """Reading H-4: targets outside [0, V) carry no loss and the mean runs over the counted tokens.  Pins: (i) the result
    equals the oracle run on the counted rows alone (loss, dg, dW) with zero dx rows where ignored -- a token's loss term
    touches only its own row of x; (ii) torch float64 cross_entropy(ignore_index=-100) under autograd; (iii) all ignored:
    zero loss and gradients; (iv) no ignored target: identical to the plain mean of H-2."""
    import torch
    import torch.nn.functional as F
    x, g, w, y = _case(8, T=20, H=24, V=50)
    yi = y.copy()
    yi[[0, 3, 4, 11, 19]] = -100
    yi[7] = 50                                       # >= V: not counted either
    keep = (yi >= 0) & (yi < 50)
    out = Hd.head_loss_fwd_bwd(x, g, w, yi, EPS)
    sub = Hd.head_loss_fwd_bwd(x[keep], g, w, yi[keep], EPS)
    assert out["loss"] == pytest.approx(sub["loss"], rel=1e-14)
    np.testing.assert_allclose(out["dx"][keep], sub["dx"], rtol=1e-12, atol=1e-16)
    assert not np.any(out["dx"][~keep])
    np.testing.assert_allclose(out["dg_final"], sub["dg_final"], rtol=1e-12, atol=1e-16)
    np.testing.assert_allclose(out["dw_head"], sub["dw_head"], rtol=1e-12, atol=1e-16)
    yt = yi.copy(); yt[7] = -100
    tx = torch.tensor(x, requires_grad=True); tg = torch.tensor(g, requires_grad=True); tw = torch.tensor(w, requires_grad=True)
    loss = F.cross_entropy(F.linear(F.rms_norm(tx, (x.shape[1],), tg, EPS), tw), torch.tensor(yt), ignore_index=-100)
    loss.backward()
    assert out["loss"] == pytest.approx(float(loss.detach()), rel=1e-13)
    np.testing.assert_allclose(out["dx"], tx.grad.numpy(), rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(out["dw_head"], tw.grad.numpy(), rtol=1e-10, atol=1e-15)
    none = Hd.head_loss_fwd_bwd(x, g, w, np.full_like(y, -1), EPS)
    assert none["loss"] == 0.0 and not np.any(none["dx"]) and not np.any(none["dw_head"]) and not np.any(none["dg_final"])
    full = Hd.head_loss_fwd_bwd(x, g, w, y, EPS)
    z = (x / np.sqrt(np.mean(x * x, axis=1) + EPS)[:, None] * g) @ w.T
    assert full["loss"] == pytest.approx(float(np.mean(full["lse"] - z[np.arange(20), y])), rel=1e-14)


def test_embed_bwd():
    rng = np.random.default_rng(7)
    ids = np.array([3, 1, 3, 0, 1, 3, 6])
    d = rng.standard_normal((7, 5))
    dE = Hd.embed_bwd(ids, d, 8)
    np.testing.assert_array_equal(dE[3], (d[0] + d[2]) + d[5])       # increasing-t order
    np.testing.assert_array_equal(dE[1], d[1] + d[4])
    np.testing.assert_array_equal(dE[0], d[3]); np.testing.assert_array_equal(dE[6], d[6])
    assert not np.any(dE[[2, 4, 5, 7]])
    np.testing.assert_allclose(np.sum(dE, axis=0), np.sum(d, axis=0), rtol=1e-13)     # nothing lost, nothing invented
    # adjoint of the gather: <dE, E> = <dx0, E[ids]> for any table E
    E = rng.standard_normal((8, 5))
    assert float(np.sum(dE * E)) == pytest.approx(float(np.sum(d * E[ids])), rel=1e-13)
