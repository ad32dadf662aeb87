"""Pins of oracle/train_oracle.py: mask (eq. 21-24), L_sparse / L_covt
(eq. 26-27), compact-model decode (L209, L501) and the Adam update ([23]'s optimiser, L324).  Each pin is
something other than the function itself: a closed form, central differences of the LOSS, the float64 C++ renderer,
a library routine (torch.optim.Adam, numpy fancy indexing / float16), or numbers worked out by hand."""
import numpy as np
import torch

import oracle
from oracle import train_oracle as T
from helpers import make_oracle, oracle_for, run_pre
from paper_2412_20720_b200 import scenes


def _rand(N, seed):
    r = np.random.default_rng(seed)
    return r.normal(-1, 0.5, (N, 4)), r.normal(size=(N, 4)), r.normal(size=(N, 4)), r.normal(size=N)


# ---- eq. 27 -------------------------------------------------------------------------------------------------
def test_sigma44_matches_the_cpp_oracle_and_closed_forms():
    sc = scenes.tiny()
    o = oracle_for(sc)
    for i in (0, 7, 100, 255):
        _, Sigma = o.rot_cov(i)
        assert abs(T.sigma44(sc.log_scale[i], sc.quat_l[i], sc.quat_r[i]) - Sigma[3, 3]) < 1e-13 * max(1, Sigma[3, 3])
    ident = np.array([1.0, 0, 0, 0])
    ls = np.array([-1.0, -2.0, 0.3, -0.7])
    assert abs(T.sigma44(ls, ident, ident) - np.exp(2 * -0.7)) < 1e-15            # R = I  =>  Sigma_44 = s_t^2
    # q_r = (a, b, c, -d) is a pure spatial rotation: time decouples, Sigma_44 = s_t^2 again
    ql = np.array([0.3, -0.5, 0.7, 0.2])
    assert abs(T.sigma44(ls, ql, ql * np.array([1, 1, 1, -1])) - np.exp(-1.4)) < 1e-14
    # q_l = e_0, q_r = (0,0,1,0): the time row of R(q_r) is (0,1,0,0), i.e. the y axis is turned onto t => Sigma_44 = s_y^2
    assert abs(T.sigma44(ls, ident, np.array([0, 0, 1.0, 0])) - np.exp(2 * -2.0)) < 1e-15


def test_covt_closed_form_identity_rotation():
    ls = np.array([[0.0, 0.0, 0.0, np.log(0.5)], [0.0, 0.0, 0.0, np.log(2.0)]])
    q = np.tile([1.0, 0, 0, 0], (2, 1))
    L, G = T.regularizers(ls, q, q)
    assert abs(L["covt"] - 0.5 * (np.exp(-0.25) + np.exp(-4.0))) < 1e-15           # eq. 27 with Sigma_44 = s_t^2
    # d/dlog s_t of exp(-s_t^2)/N = -2 s_t^2 exp(-s_t^2)/N; the spatial scales do not enter
    np.testing.assert_allclose(G["log_scale"][:, 3], [-2 * 0.25 * np.exp(-0.25) / 2, -2 * 4 * np.exp(-4.0) / 2], rtol=1e-14)
    assert np.abs(G["log_scale"][:, :3]).max() == 0
    assert L["sparse"] == 0 and np.abs(G["quat_l"]).max() < 1e-16                   # sign(0) = 0, Sigma_44 stationary


# ---- eq. 26 -------------------------------------------------------------------------------------------------
def test_sparse_closed_forms():
    ls = np.zeros((3, 4))
    ql = np.array([[1.0, 0, 0, 0], [2.0, 0, 0, 0], [1.0, 1.0, 0, 0]])
    qr = np.array([[0, 1.0, 0, 0], [0.5, 0, 0, 0], [1.0, -1.0, 0, 0]])
    L, _ = T.regularizers(ls, ql, qr, lambda_covt=0.0)
    # |e0 - e1|_1 = 2;  normalised (2,0,0,0) and (0.5,0,0,0) coincide -> 0;  (1,1)/sqrt2 - (1,-1)/sqrt2 -> sqrt2
    assert abs(L["sparse"] - (2.0 + 0.0 + np.sqrt(2.0)) / 3) < 1e-15
    L2, _ = T.regularizers(ls, 3.7 * ql, 0.2 * qr, lambda_covt=0.0)                  # T1: scale of the parameters is irrelevant
    assert abs(L2["sparse"] - L["sparse"]) < 1e-15


def test_regularizer_gradients_match_central_differences_of_the_losses():
    ls, ql, qr, m = _rand(6, 1)
    lam = dict(lambda_sparse=0.7, lambda_covt=1.3, lambda_mask=0.5)
    _, G = T.regularizers(ls, ql, qr, m, **lam)

    def total(a):
        L, _ = T.regularizers(a["log_scale"], a["quat_l"], a["quat_r"], a["mask_logit"])
        return 0.7 * L["sparse"] + 1.3 * L["covt"] + 0.5 * L["mask"]

    base = dict(log_scale=ls, quat_l=ql, quat_r=qr, mask_logit=m)
    h = 1e-6
    for name, arr in base.items():
        fd = np.zeros_like(arr)
        for idx in np.ndindex(arr.shape):
            up, dn = dict(base), dict(base)
            up[name] = arr.copy(); up[name][idx] += h
            dn[name] = arr.copy(); dn[name][idx] -= h
            fd[idx] = (total(up) - total(dn)) / (2 * h)
        assert np.abs(fd - G[name]).max() <= 1e-7 * np.abs(fd).max(), name
    # quaternions are normalised inside: the gradient is orthogonal to the parameter
    assert np.abs((G["quat_l"] * ql).sum(1)).max() < 1e-15 and np.abs((G["quat_r"] * qr).sum(1)).max() < 1e-15


# ---- eq. 21-24 ----------------------------------------------------------------------------------------------
def test_mask_values_and_mask_loss():
    m = np.array([-5.0, -0.1, 0.0, 0.1, 5.0])
    np.testing.assert_array_equal(T.mask_hat(m, 0.5), [0, 0, 0, 1, 1])                # 1{Sigmoid(m) > eps}, strict
    np.testing.assert_array_equal(T.mask_hat(m, 0.01), [0, 1, 1, 1, 1])               # Sigmoid(-5) = 0.0067
    S, a = T.masked_scale_opacity(np.zeros((5, 4)), np.zeros(5), m, 0.5)
    np.testing.assert_array_equal(S[:, 0], [0, 0, 0, 1, 1])
    np.testing.assert_array_equal(a, [0, 0, 0, 0.5, 0.5])
    L, G = T.regularizers(np.zeros((5, 4)), np.tile([1.0, 0, 0, 0], (5, 1)), np.tile([1.0, 0, 0, 0], (5, 1)), m)
    assert abs(L["mask"] - np.mean(1 / (1 + np.exp(-m)))) < 1e-16                    # eq. 24
    assert abs(G["mask_logit"][2] - 0.25 / 5) < 1e-16                                # Sigmoid'(0) = 1/4


def test_mask_gradient_is_the_derivative_of_the_render_wrt_a_common_factor_on_scale_and_opacity():
    """eq. 22-23: L depends on M_hat through S_hat = M_hat S and alpha_hat = M_hat alpha.  Render with the float64 C++
    oracle at M_hat = 1 +- h for ONE primitive and compare the central difference with mask_backward."""
    sc = scenes.fd_scene(5)
    view = sc.views[0]
    G = scenes.upstream_normal(5, view.width, view.height).astype(np.float64)
    cfg = dict(oracle.PURE_CFG)
    o = run_pre(make_oracle(sc), view, cfg)
    o.forward()
    g = o.backward(G)
    m = np.linspace(-1.0, 2.0, sc.N)
    eps = 0.2                                                                        # Sigmoid(-1) = 0.27 > eps: all kept
    got = T.mask_backward(m, eps, sc.opacity_logit, g["log_scale"], g["opacity_logit"])
    M = 1 / (1 + np.exp(-m))
    h = 1e-6
    for i in range(sc.N):
        vals = []
        for Mh in (1 + h, 1 - h):
            s2 = sc.subset(list(range(sc.N)))
            s2.log_scale, s2.opacity_logit = s2.log_scale.astype(np.float64), s2.opacity_logit.astype(np.float64)
            s2.log_scale[i] = s2.log_scale[i] + np.log(Mh)                            # s_hat = M_hat s
            a = Mh / (1 + np.exp(-s2.opacity_logit[i]))                               # alpha_hat = M_hat alpha
            s2.opacity_logit[i] = np.log(a / (1 - a))
            oo = run_pre(make_oracle(s2), view, cfg)
            img = oo.forward()[0]
            vals.append(float((img * G).sum()))
        fd = (vals[0] - vals[1]) / (2 * h) * M[i] * (1 - M[i])                         # eq. 21: dM_hat/dm = M (1 - M)
        assert abs(fd - got[i]) <= 2e-5 * max(abs(fd), 1e-3), (i, fd, got[i])
    # a masked primitive gets nothing from the render
    assert T.mask_backward(np.array([-3.0]), 0.2, np.zeros(1), np.ones((1, 4)), np.ones(1))[0] == 0


# ---- compact model decode -------------------------------------------------------------------------------------
def test_rvq_decode_is_a_sum_of_table_lookups():
    r = np.random.default_rng(3)
    cb = r.normal(size=(6, 64, 4))
    idx = r.integers(0, 64, size=(50, 6))
    want = sum(cb[s][idx[:, s]] for s in range(6))                                    # numpy fancy indexing per stage
    np.testing.assert_allclose(T.rvq_decode(idx, cb), want, rtol=0, atol=1e-15)
    # hand-worked: two stages, entries (1, 2) and (0.25, -0.5)
    cb2 = np.array([[[0.0, 0.0], [1.0, 2.0]], [[0.25, -0.5], [9.0, 9.0]]])
    np.testing.assert_array_equal(T.rvq_decode(np.array([[1, 0]]), cb2), [[1.25, 1.5]])


def test_half_precision_and_minmax_values():
    c = dict(mean_f16=np.array([[0.1, 1.0 / 3.0, -2.5, 1000.3]], dtype=np.float16), opacity_code=np.array([51], dtype=np.uint8),
             opacity_lo=-4.0, opacity_hi=6.0, scale_idx=np.zeros((1, 1), dtype=np.uint8), scale_cb=np.zeros((1, 1, 4)),
             rot_l_idx=np.zeros((1, 1), dtype=np.uint8), rot_r_idx=np.zeros((1, 1), dtype=np.uint8),
             rot_cb=np.array([[[1.0, 0, 0, 0]]]), dc_idx=np.zeros((1, 1), dtype=np.uint8), dc_cb=np.array([[[0.5, 0.25, 0.125]]]),
             rest_idx=None, rest_cb=None)
    d = T.decode_compact(c)
    # binary16 neighbours of 0.1, 1/3 and 1000.3 (11-bit significand): 0.0999755859375, 0.333251953125, 1000.5
    np.testing.assert_array_equal(d["mean"], [[0.0999755859375, 0.333251953125, -2.5, 1000.5]])
    assert abs(d["opacity_logit"][0] - (-4.0 + 0.2 * 10.0)) < 1e-15                   # code 51 / 255 = 0.2
    assert T.minmax_dequant(0, -4, 6) == -4 and T.minmax_dequant(255, -4, 6) == 6
    assert d["sh"].shape == (1, 1, 3) and d["sh"][0, 0, 2] == 0.125


def test_decode_compact_layout_of_rest_coefficients():
    r = np.random.default_rng(5)
    N, K = 7, 8
    c = scenes_free_compact(r, N, K)
    d = T.decode_compact(c)
    i = 3
    want_rest = sum(c["rest_cb"][s, c["rest_idx"][i, s]] for s in range(c["rest_cb"].shape[0]))
    np.testing.assert_allclose(d["sh"][i, 1:, :].ravel(), want_rest, atol=1e-15)      # coefficient-major, channel last
    np.testing.assert_allclose(d["sh"][i, 0, :], sum(c["dc_cb"][s, c["dc_idx"][i, s]] for s in range(6)), atol=1e-15)
    np.testing.assert_allclose(d["quat_r"][i], sum(c["rot_cb"][s, c["rot_r_idx"][i, s]] for s in range(6)), atol=1e-15)


def scenes_free_compact(r, N, K):
    return dict(mean_f16=r.normal(size=(N, 4)).astype(np.float16), opacity_code=r.integers(0, 256, N).astype(np.uint8),
                opacity_lo=-3.0, opacity_hi=5.0, scale_idx=r.integers(0, 64, (N, 6)).astype(np.uint8),
                scale_cb=r.normal(size=(6, 64, 4)), rot_l_idx=r.integers(0, 64, (N, 6)).astype(np.uint8),
                rot_r_idx=r.integers(0, 64, (N, 6)).astype(np.uint8), rot_cb=r.normal(size=(6, 64, 4)),
                dc_idx=r.integers(0, 64, (N, 6)).astype(np.uint8), dc_cb=r.normal(size=(6, 64, 3)),
                rest_idx=r.integers(0, 256, (N, 8)).astype(np.uint8), rest_cb=r.normal(size=(8, 256, (K - 1) * 3)))


# ---- Adam ---------------------------------------------------------------------------------------------------
def test_adam_matches_torch_and_closed_forms():
    r = np.random.default_rng(7)
    p0 = r.normal(size=20)
    grads = [r.normal(size=20) * (10.0 ** r.integers(-4, 2)) for _ in range(6)]
    tp = torch.tensor(p0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([tp], lr=1.6e-3, betas=(0.9, 0.999), eps=1e-15)
    p, m, v = p0.copy(), np.zeros(20), np.zeros(20)
    for step, g in enumerate(grads, start=1):
        tp.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        p, m, v = T.adam_step(p, g, m, v, step, 1.6e-3)
        np.testing.assert_allclose(p, tp.detach().numpy(), rtol=1e-12, atol=1e-15)
    # first step: m_hat = g, v_hat = g^2  =>  p1 = p0 - lr sign(g) (eps negligible)
    g = np.array([3.0, -0.02, 0.0])
    p1, m1, v1 = T.adam_step(np.zeros(3), g, np.zeros(3), np.zeros(3), 1, 0.01)
    np.testing.assert_allclose(p1, [-0.01, 0.01, 0.0], atol=1e-14)
    np.testing.assert_allclose(m1, 0.1 * g)
    np.testing.assert_allclose(v1, 0.001 * g * g)
    # constant gradient: bias correction makes every step exactly lr sign(g)
    p, m, v = np.zeros(1), np.zeros(1), np.zeros(1)
    for step in range(1, 8):
        p, m, v = T.adam_step(p, np.array([0.3]), m, v, step, 0.01)
    assert abs(p[0] + 0.07) < 1e-12
