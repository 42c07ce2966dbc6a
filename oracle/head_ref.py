"""head_ref -- fp64 CPU oracle of the steps either side of the decoder stack: the final
RMSNorm, the LM-head projection, the next-token cross-entropy loss with its gradients, and the embedding backward.

TEST INFRASTRUCTURE ONLY (same rules as lspref.py): only ``tests/`` may import it; it shares no code with the CUDA
path and imports nothing from ``paper_2510_02483_b200/``.

What the paper fixes: "pre-training" of a Llama model with a 32000-entry vocabulary and the
standard Llama components; its FLOP accounting includes the LM head and excludes the embedding lookup
(SURVEY.md Appendix A).  It prints no loss definition, so the readings are the standard ones:
  H-1  the model ends with an RMSNorm (gain g_final, same eps as the layers, reading A-3) and a bias-free LM head
       W_head [V, H] ([out, in] like every projection, reading A-9; not tied to the embedding);
  H-2  loss = mean over the T tokens of the natural-log cross-entropy of softmax(logits_t) against target id y_t;
  H-3  the embedding gradient is the scatter-add of the gradient rows: dE[v,:] = sum over {t : id_t = v} of dx0[t,:];
  H-4  a target outside [0, V) (e.g. -100: padding, or the last token of each sequence of a packed SFT / DPO batch,
       PAPER.md:176-186) carries no loss: the mean of H-2 runs over the n COUNTED tokens only (the convention of
       torch.nn.functional.cross_entropy(ignore_index=...)); with every target counted this is H-2 unchanged.
Plain numpy float64, one statement per formula; numpy.matmul is the only library primitive.
"""
from __future__ import annotations

import numpy as np

F64 = np.float64


def head_loss_fwd_bwd(x, g_final, w_head, targets, eps):
    """x [T,H], g_final [H], w_head [V,H], targets int [T].  Returns dict(loss, lse [T], dx [T,H], dg_final [H], dw_head [V,H]).

    r_t = 1/sqrt(mean_j x_tj^2 + eps);  xn = x r g_final                                   (H-1, A-3)
    z = xn W_head^T;  lse_t = m_t + log sum_v exp(z_tv - m_t), m_t = max_v z_tv;  loss = mean_t (lse_t - z_t,y_t)   (H-2)
    dz_tv = (exp(z_tv - lse_t) - [v = y_t]) / T;  dW_head = dz^T xn;  dxn = dz W_head;  then the RMSNorm backward.
    H-4: the mean and the 1/T run over the n tokens whose target lies in [0, V); the other rows of dz are zero
    (n = 0: loss 0, all gradients 0).
    """
    x = np.asarray(x, F64); g_final = np.asarray(g_final, F64); w_head = np.asarray(w_head, F64)
    y = np.asarray(targets, np.int64)
    T = x.shape[0]
    r = 1.0 / np.sqrt(np.mean(x * x, axis=1) + eps)
    n = x * r[:, None]
    xn = n * g_final[None, :]
    z = np.matmul(xn, w_head.T)
    m = np.max(z, axis=1)
    lse = m + np.log(np.sum(np.exp(z - m[:, None]), axis=1))
    counted = (y >= 0) & (y < w_head.shape[0])
    tc = np.arange(T)[counted]
    n_counted = int(tc.size)
    loss = float(np.sum(lse[tc] - z[tc, y[tc]]) / n_counted) if n_counted else 0.0
    dz = np.exp(z - lse[:, None])
    dz[tc, y[tc]] -= 1.0
    dz[~counted, :] = 0.0
    dz /= max(n_counted, 1)
    dw_head = np.matmul(dz.T, xn)
    dxn = np.matmul(dz, w_head)
    dn = dxn * g_final[None, :]
    dx = r[:, None] * (dn - n * np.mean(dn * n, axis=1)[:, None])
    dg_final = np.sum(dxn * n, axis=0)
    return dict(loss=loss, lse=lse, dx=dx, dg_final=dg_final, dw_head=dw_head)


def embed_bwd(ids, dx0, vocab):
    """dE [vocab, H]: dE[v,:] = sum over {t : id_t = v} dx0[t,:], tokens added in increasing t (H-3)."""
    ids = np.asarray(ids, np.int64); dx0 = np.asarray(dx0, F64)
    dE = np.zeros((vocab, dx0.shape[1]), F64)
    for t in range(ids.shape[0]):
        dE[ids[t], :] += dx0[t, :]
    return dE
