"""float64 numpy ORACLE for the per-primitive training-side terms next to the rasterizer.

TEST INFRASTRUCTURE ONLY (same rule as the rest of ``oracle/``): only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s CPU legs may import it.  It shares nothing with ``paper_2412_20720_b200/csrc`` and never imports the
product package.  Everything is float64 and written in the paper's order; PAPER.md:L<line> citations.

What it states
  * eq. 21-24: the learnable mask, its straight-through gradient and the mask loss;
  * eq. 26 (L239): L_sparse, eq. 27 (L245): L_covt, with analytic gradients (pinned by central differences and
    closed forms in tests/test_oracle_train_pins.py);
  * the decode of the compact model of section 4.2 / 8.3.1 (L209, L501): residual vector quantisation = sum of one
    codebook entry per stage, half-precision positions, k-bit min-max opacity;
  * one Adam update (the optimiser of [23] whose settings the paper adopts, L324) — textbook Kingma & Ba.

Readings where the paper is silent (T1-T6) are repeated at each function.
Parity unpinned by the paper (conventions only): T1 (which norm / which quaternions in eq. 26), T4 (what the
codebooks and the quantisers store), T6 (Adam hyper-parameters).  The formulas themselves are pinned.
"""
from __future__ import annotations

import numpy as np


# ---------------------------------------------------------------------------------------------------------------
# eq. 8 (sign pattern de-garbled as DESIGN.md G1): left / right isoclinic matrices.
# Both are LINEAR in the quaternion, so d(matrix)/d(q_i) = matrix(e_i): used for the gradients below.
def left_matrix(q):
    a, b, c, d = q
    return np.array([[a, -b, -c, -d], [b, a, -d, c], [c, d, a, -b], [d, -c, b, a]], dtype=np.float64)


def right_matrix(q):
    p, qq, r, s = q
    return np.array([[p, -qq, -r, -s], [qq, p, s, -r], [r, -s, p, qq], [s, r, -qq, p]], dtype=np.float64)


def _normalise_vjp(q, g_hat):
    """q_hat = q / |q|  =>  dL/dq = (g_hat - q_hat (q_hat . g_hat)) / |q|."""
    n = np.linalg.norm(q)
    qh = q / n
    return (g_hat - qh * np.dot(qh, g_hat)) / n


def sigmoid(x):
    x = np.asarray(x, dtype=np.float64)
    return np.where(x >= 0, 1.0 / (1.0 + np.exp(-np.abs(x))), np.exp(-np.abs(x)) / (1.0 + np.exp(-np.abs(x))))


# ---------------------------------------------------------------------------------------------------------------
def sigma44(log_scale_i, quat_l_i, quat_r_i):
    """Sigma_44 of one primitive: last diagonal entry of R S S^T R^T (eq. 7), R = L(q_l) R(q_r) (eq. 8)."""
    s = np.exp(np.asarray(log_scale_i, dtype=np.float64))
    ql = np.asarray(quat_l_i, dtype=np.float64)
    qr = np.asarray(quat_r_i, dtype=np.float64)
    R = left_matrix(ql / np.linalg.norm(ql)) @ right_matrix(qr / np.linalg.norm(qr))
    Sigma = R @ np.diag(s * s) @ R.T
    return Sigma[3, 3]


def regularizers(log_scale, quat_l, quat_r, mask_logit=None, lambda_sparse=1.0, lambda_covt=1.0, lambda_mask=1.0):
    """L_sparse (eq. 26), L_covt (eq. 27), L_mask (eq. 24) and the gradient of
    lambda_sparse L_sparse + lambda_covt L_covt + lambda_mask L_mask  w.r.t. log_scale, quat_l, quat_r, mask_logit.

    Readings: T1 — q_l, q_r in eq. 26 are the paper's (unit) quaternions, i.e. the normalised parameters, and the
    norm is the 1-norm ("an L1 loss on the difference between its q_l and q_r", L237); sign(0) = 0.
    T2 — Sigma_44 in eq. 27 is the (4,4) entry of eq. 7 with s = exp(log_scale).  Means are over all N primitives.
    Returns (losses dict, grads dict)."""
    ls = np.asarray(log_scale, dtype=np.float64)
    QL = np.asarray(quat_l, dtype=np.float64)
    QR = np.asarray(quat_r, dtype=np.float64)
    N = ls.shape[0]
    g_ls, g_ql, g_qr = np.zeros((N, 4)), np.zeros((N, 4)), np.zeros((N, 4))
    L_sparse = L_covt = 0.0
    E = np.eye(4)
    for i in range(N):
        s = np.exp(ls[i])
        nl, nr = np.linalg.norm(QL[i]), np.linalg.norm(QR[i])
        qlh, qrh = QL[i] / nl, QR[i] / nr
        # eq. 26
        diff = qlh - qrh
        L_sparse += np.abs(diff).sum() / N
        gh_l = lambda_sparse * np.sign(diff) / N
        gh_r = -lambda_sparse * np.sign(diff) / N
        # eq. 27
        Lm, Rm = left_matrix(qlh), right_matrix(qrh)
        R = Lm @ Rm
        S44 = float(np.sum((R[3, :] * s) ** 2))
        e = np.exp(-S44)
        L_covt += e / N
        gS = -lambda_covt * e / N                       # dL/dSigma_44
        g_ls[i] += gS * 2.0 * (R[3, :] * s) ** 2        # d Sigma_44 / d log s_k = 2 (R_4k s_k)^2
        G = np.zeros((4, 4))
        G[3, :] = gS * 2.0 * R[3, :] * s * s            # dL/dR (only the time row of R enters Sigma_44)
        GL, GR = G @ Rm.T, Lm.T @ G                     # R = Lm Rm
        for k in range(4):
            gh_l[k] += np.sum(GL * left_matrix(E[k]))
            gh_r[k] += np.sum(GR * right_matrix(E[k]))
        g_ql[i] += _normalise_vjp(QL[i], gh_l)
        g_qr[i] += _normalise_vjp(QR[i], gh_r)
    losses = dict(sparse=L_sparse, covt=L_covt, mask=0.0)
    grads = dict(log_scale=g_ls, quat_l=g_ql, quat_r=g_qr, mask_logit=None)
    if mask_logit is not None:
        M = sigmoid(mask_logit)                         # eq. 24: L_mask = mean_i M_i,  M = Sigmoid(m) (L215)
        losses["mask"] = float(M.mean())
        # dM/dm = M (1 - M), evaluated as Sigmoid(m) Sigmoid(-m): the same quantity without the cancellation of 1 - M for
        # saturated m (|m| > 37 rounds M to exactly 0 or 1 in float64)
        grads["mask_logit"] = lambda_mask * M * sigmoid(-np.asarray(mask_logit, dtype=np.float64)) / N
    return losses, grads


# ---------------------------------------------------------------------------------------------------------------
# eq. 21-23: learnable mask.  M = Sigmoid(m); M_hat = stop_gradient(1{M > eps} - M) + M, i.e.
# the VALUE of M_hat is the indicator and dM_hat/dM = 1;  S_hat = M_hat S (all four scales), alpha_hat = M_hat alpha.
def mask_hat(mask_logit, eps):
    """Forward value of eq. 21."""
    return (sigmoid(mask_logit) > eps).astype(np.float64)


def masked_scale_opacity(log_scale, opacity_logit, mask_logit, eps):
    """eq. 22-23 in value space: (S_hat [N,4], alpha_hat [N])."""
    Mh = mask_hat(mask_logit, eps)
    return Mh[:, None] * np.exp(np.asarray(log_scale, dtype=np.float64)), Mh * sigmoid(opacity_logit)


def mask_backward(mask_logit, eps, opacity_logit, g_log_scale, g_opacity_logit):
    """dL/dm from the gradients the renderer returned for a kept primitive (M_hat = 1).
    L depends on M_hat through s_hat_k = M_hat s_k and alpha_hat = M_hat alpha, so at M_hat = 1
        dL/dM_hat = sum_k dL/ds_hat_k s_k + dL/dalpha_hat alpha
                  = sum_k dL/dlog s_k       + dL/dlogit / (1 - alpha)          (alpha' = alpha (1 - alpha)),
    and by eq. 21 dM_hat/dm = dM/dm = M (1 - M).
    Reading T3: a masked primitive (M_hat = 0) has alpha_hat = 0 and a degenerate covariance — it is removed from the
    render, receives no rendering gradient (the inputs g_* are zero for it) and only L_mask acts on its m."""
    M = sigmoid(mask_logit)
    Mh = mask_hat(mask_logit, eps)
    one_minus = sigmoid(-np.asarray(opacity_logit, dtype=np.float64))      # 1 - alpha
    dL_dMhat = np.asarray(g_log_scale, dtype=np.float64).sum(axis=1) + np.asarray(g_opacity_logit, dtype=np.float64) / one_minus
    return Mh * dL_dMhat * M * sigmoid(-np.asarray(mask_logit, dtype=np.float64))      # M (1 - M) without cancellation


# ---------------------------------------------------------------------------------------------------------------
# Compact model decode (section 4.2; sizes L501: scale 6 codebooks x 64 entries, both quaternions share
# 6 x 64, base colour 6 x 64, rest of the 4DSH coefficients 8 x 256; positions half precision; opacity 8-bit min-max).
# Reading T4: a codebook entry has the shape of the STORED parameter it replaces (log-scale [4], raw quaternion [4],
# coefficient k = 0 [3], coefficients k = 1..K-1 [(K-1)*3]); residual VQ decodes to the SUM over stages of the indexed
# entries; the min-max quantiser stores the opacity logit as  lo + code (hi - lo) / (2^bits - 1).  Huffman coding of
# the indices (L209) is a lossless file format and not part of the render path.
def rvq_decode(indices, codebooks):
    """indices [N,S] integer, codebooks [S,E,D] -> [N,D] = sum_s codebooks[s, indices[:,s], :]."""
    idx = np.asarray(indices)
    cb = np.asarray(codebooks, dtype=np.float64)
    out = np.zeros((idx.shape[0], cb.shape[2]))
    for n in range(idx.shape[0]):
        for s in range(cb.shape[0]):
            out[n] += cb[s, int(idx[n, s])]
    return out


def minmax_dequant(code, lo, hi, bits=8):
    return float(lo) + np.asarray(code, dtype=np.float64) * (float(hi) - float(lo)) / float(2 ** bits - 1)


def decode_compact(c):
    """c: dict with mean_f16 [N,4] float16, opacity_code [N] uint8, opacity_lo/hi, scale_idx [N,S1], scale_cb,
    rot_l_idx, rot_r_idx [N,S2], rot_cb, dc_idx [N,S3], dc_cb [S3,E,3], rest_idx [N,S4], rest_cb [S4,E',(K-1)*3] (or
    None when K = 1).  Returns the six parameter arrays of the full model in float64."""
    N = c["mean_f16"].shape[0]
    mean = np.asarray(c["mean_f16"], dtype=np.float16).astype(np.float64)
    log_scale = rvq_decode(c["scale_idx"], c["scale_cb"])
    quat_l = rvq_decode(c["rot_l_idx"], c["rot_cb"])
    quat_r = rvq_decode(c["rot_r_idx"], c["rot_cb"])
    logit = minmax_dequant(c["opacity_code"], c["opacity_lo"], c["opacity_hi"], c.get("opacity_bits", 8))
    dc = rvq_decode(c["dc_idx"], c["dc_cb"])
    if c.get("rest_cb") is not None:
        rest = rvq_decode(c["rest_idx"], c["rest_cb"])
        sh = np.concatenate([dc, rest], axis=1).reshape(N, -1, 3)
    else:
        sh = dc.reshape(N, 1, 3)
    return dict(mean=mean, log_scale=log_scale, quat_l=quat_l, quat_r=quat_r, opacity_logit=logit, sh=sh)


# ---------------------------------------------------------------------------------------------------------------
# One Adam update (Kingma & Ba 2015, Algorithm 1) — the optimiser of [23], whose settings the paper adopts (L324).
# Reading T6: beta1 = 0.9, beta2 = 0.999, eps = 1e-15 ([23]'s values), bias-corrected, no weight decay; the update is
# dense (every primitive moves by its momentum even when its gradient of this step is zero).
def adam_step(p, g, m, v, step, lr, beta1=0.9, beta2=0.999, eps=1e-15):
    p, g, m, v = (np.asarray(a, dtype=np.float64) for a in (p, g, m, v))
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    m_hat = m / (1.0 - beta1 ** step)
    v_hat = v / (1.0 - beta2 ** step)
    p = p - lr * m_hat / (np.sqrt(v_hat) + eps)
    return p, m, v
