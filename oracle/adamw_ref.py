"""adamw_ref -- the fp64 CPU oracle of the optimizer step that follows the layer backward.

TEST INFRASTRUCTURE ONLY (same rules as lspref.py): only ``tests/`` may import it; it shares no code with the CUDA
path and imports nothing from ``paper_2510_02483_b200/``.

What the paper fixes (section 2.5.2; section 2.5.3; Table 2):
AdamW [40] with beta1 = 0.90, beta2 = 0.95, weight decay 0.01, gradient clipping threshold 1.0; cosine learning-rate
schedule, maximum 1.2e-3, minimum 1.0e-5, 2000 warm-up steps; BF16 mixed precision.  It gives no equation, so the
formulas are those of the cited reference [40] (decoupled weight decay, bias-corrected moments) in the readings listed
in DESIGN.md section 12:
  O-1  epsilon = 1e-8, added to sqrt(v_hat) (the reference's Algorithm 2);
  O-2  clipping is by the GLOBAL l2 norm over all tensors of the call: g <- g * min(1, clip / (norm + 1e-6));
  O-3  warm-up is linear from 0: lr(t) = lr_max * t / warmup for 1 <= t <= warmup; then
       lr(t) = lr_min + (lr_max - lr_min)/2 * (1 + cos(pi * (t - warmup) / (total - warmup))), lr_min after `total`
       (the paper does not state the total number of steps: it is a parameter);
  O-4  weight decay applies to tensors flagged `decay` (the 2-D projection weights), not to the RMSNorm gains;
  O-5  mixed precision = fp32 master weights and moments; the bf16 model weight is the round-to-nearest-even of the
       updated master weight.
Every function is plain float64 numpy, one statement per formula.
"""
from __future__ import annotations

import math

import numpy as np

# Table 2
BETA1, BETA2, WEIGHT_DECAY, CLIP_NORM = 0.90, 0.95, 0.01, 1.0
LR_MAX, LR_MIN, WARMUP = 1.2e-3, 1.0e-5, 2000
EPS = 1e-8          # reading O-1


def lr_cosine(step: int, lr_max: float = LR_MAX, lr_min: float = LR_MIN, warmup: int = WARMUP, total: int = 100000) -> float:
    """Learning rate of optimizer step `step` (1-based), reading O-3."""
    if step <= warmup:
        return lr_max * step / warmup
    if step >= total:
        return lr_min
    return lr_min + 0.5 * (lr_max - lr_min) * (1.0 + math.cos(math.pi * (step - warmup) / (total - warmup)))


def global_grad_norm(grads) -> float:
    """l2 norm over every element of every tensor (reading O-2)."""
    return math.sqrt(sum(float(np.sum(np.asarray(g, np.float64) ** 2)) for g in grads))


def clip_coefficient(norm: float, clip: float = CLIP_NORM) -> float:
    return min(1.0, clip / (norm + 1e-6))


def adamw_step(params, grads, ms, vs, decay_flags, step: int, lr: float, beta1: float = BETA1, beta2: float = BETA2,
               eps: float = EPS, weight_decay: float = WEIGHT_DECAY, clip: float = CLIP_NORM):
    """One AdamW step with global-norm clipping on lists of float64 arrays.  Returns (new_params, new_ms, new_vs, norm).

    m <- beta1 m + (1 - beta1) g ;  v <- beta2 v + (1 - beta2) g^2           (g already clipped)
    m_hat = m / (1 - beta1^t) ;     v_hat = v / (1 - beta2^t)
    p <- p - lr * ( m_hat / (sqrt(v_hat) + eps) + weight_decay * p )          (ref [40], Algorithm 2; O-1, O-4)
    """
    norm = global_grad_norm(grads)
    c = clip_coefficient(norm, clip)
    out_p, out_m, out_v = [], [], []
    for p, g, m, v, dec in zip(params, grads, ms, vs, decay_flags):
        p = np.asarray(p, np.float64); m = np.asarray(m, np.float64); v = np.asarray(v, np.float64)
        g = np.asarray(g, np.float64) * c
        m_new = beta1 * m + (1.0 - beta1) * g
        v_new = beta2 * v + (1.0 - beta2) * g * g
        m_hat = m_new / (1.0 - beta1 ** step)
        v_hat = v_new / (1.0 - beta2 ** step)
        wd = weight_decay if dec else 0.0
        p_new = p - lr * (m_hat / (np.sqrt(v_hat) + eps) + wd * p)
        out_p.append(p_new); out_m.append(m_new); out_v.append(v_new)
    return out_p, out_m, out_v, norm


def bf16_rne(x) -> np.ndarray:
    """float64 -> nearest bfloat16 (ties to even), returned as float64 values (reading O-5).  Written from the format
    definition (8 exponent bits, 7 fraction bits): round the float32 bit pattern to its upper 16 bits."""
    f = np.asarray(x, np.float64).astype(np.float32)
    u = f.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).astype(np.float64)
