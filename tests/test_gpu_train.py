"""GPU parity of the training-side entry points (fdgs_mask_apply, fdgs_regularizers, fdgs_adam_step,
fdgs_decode_compact) against oracle/train_oracle.py and the float64 renderer, through the C ABI.
Tolerances: gradients rel-L2 <= 1e-3 (north_star), losses 1e-5 relative (fp32 atomics), Adam / decode element-wise
2e-6 relative to the magnitude of the terms (fp32 arithmetic, a handful of operations), fp16 positions bit-exact."""
import numpy as np
import pytest
import torch

import oracle
from oracle import train_oracle as T
from helpers import make_oracle, rel_l2, run_pre
from paper_2412_20720_b200 import fdgs, scenes, train

pytestmark = pytest.mark.gpu


def _cuda(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t.to(dtype) if dtype is not None else t).cuda()


def _prefilled_grads(ds, seed):
    """'Rendering' gradients already accumulated: seeded noise (the entry points must add to / read them)."""
    g = ds.zero_grads()
    gen = torch.Generator(device="cpu").manual_seed(seed)
    for k in ("log_scale", "quat_l", "quat_r", "opacity_logit"):
        g[k] += (1e-4 * torch.randn(g[k].shape, generator=gen)).cuda()
    return g


@pytest.mark.parametrize("name,N", [("tiny_random_rotations", 256), ("video_tilted", 20011)])
def test_regularizers_and_mask_gradient_match_the_oracle(name, N):
    sc = scenes.tiny() if name.startswith("tiny") else scenes.multiview_video(N=N, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    g = _prefilled_grads(ds, 1)
    g0 = {k: v.cpu().numpy().astype(np.float64) for k, v in g.items() if v is not None}
    m = scenes.normal(11, 7, sc.N).astype(np.float32)                       # mask logits ~ N(0,1): about half masked at eps 0.5
    eps = 0.5
    lam = dict(lambda_sparse=0.03, lambda_covt=0.2, lambda_mask=0.0005)
    gm = torch.zeros(sc.N, device="cuda") + 0.125                           # += is checked with a non-zero start
    losses = torch.zeros(3, device="cuda")
    train.regularizers(ds, g, mask_logit=_cuda(m), mask_eps=eps, grad_mask_logit=gm, losses=losses, **lam)
    torch.cuda.synchronize()
    L, G = T.regularizers(sc.log_scale, sc.quat_l, sc.quat_r, m, **lam)
    want_m = 0.125 + G["mask_logit"] + T.mask_backward(m, eps, sc.opacity_logit, g0["log_scale"], g0["opacity_logit"])
    fragile = np.abs(T.sigmoid(m) - eps) < 1e-6                             # threshold decided in fp32 vs fp64
    got_m = gm.cpu().numpy().astype(np.float64)
    assert rel_l2(got_m[~fragile], want_m[~fragile]) < 1e-5
    for k in ("log_scale", "quat_l", "quat_r"):
        got = g[k].cpu().numpy().astype(np.float64) - g0[k]                 # what the call added
        err = rel_l2(got, G[k])
        print("PARITY", name, k, err)
        assert err < 1e-3, (k, err)
    np.testing.assert_array_equal(g["opacity_logit"].cpu().numpy().astype(np.float64), g0["opacity_logit"])   # read only
    got_L = losses.cpu().numpy().astype(np.float64)
    np.testing.assert_allclose(got_L, [L["sparse"], L["covt"], L["mask"]], rtol=1e-5)
    assert L["covt"] > 1e-3 and L["sparse"] > 1e-3


def test_regularizers_without_mask_and_degenerate_primitives():
    sc = scenes.tiny()
    sc.quat_l[3] = 0.0                                                      # zero quaternion: contributes nothing
    sc.log_scale[5, 1] = np.nan
    ds = fdgs.DeviceScene.from_scene(sc)
    g = ds.zero_grads()
    losses = torch.zeros(3, device="cuda")
    train.regularizers(ds, g, lambda_sparse=1.0, lambda_covt=1.0, losses=losses)
    torch.cuda.synchronize()
    keep = np.ones(sc.N, dtype=bool)
    keep[[3, 5]] = False
    L, G = T.regularizers(sc.log_scale[keep], sc.quat_l[keep], sc.quat_r[keep])
    scale = keep.sum() / sc.N                                               # the mean is over all N primitives
    np.testing.assert_allclose(losses.cpu().numpy()[:2], [L["sparse"] * scale, L["covt"] * scale], rtol=1e-5)
    for k in ("log_scale", "quat_l", "quat_r"):
        got = g[k].cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all() and np.abs(got[~keep]).max() == 0
        assert rel_l2(got[keep], G[k] * scale) < 1e-3
    assert losses[2].item() == 0


def test_masked_render_end_to_end_matches_the_oracle_with_masked_primitives_removed():
    """eq. 21-23 through the renderer: GPU = mask_apply -> preprocess/forward/backward -> regularizers(mask);
    oracle = the same scene WITHOUT the masked primitives (alpha_hat = 0 contributes nothing), then mask_backward."""
    sc = scenes.tiny()
    view = sc.views[0]
    m = (1.5 * scenes.normal(12, 7, sc.N)).astype(np.float32)
    eps = 0.4
    keep = T.mask_hat(m, eps).astype(bool)
    assert 60 < keep.sum() < sc.N - 20
    dL = scenes.upstream_normal(0, view.width, view.height)
    # --- GPU
    ds = fdgs.DeviceScene.from_scene(sc)
    masked = fdgs.DeviceScene(ds.sh_degree, ds.n_time, ds.mean, ds.log_scale, ds.quat_l, ds.quat_r,
                              train.mask_apply(_cuda(m), eps, ds.opacity_logit), ds.sh)
    r = fdgs.Renderer(masked, view.width, view.height, 1 << 16)
    cv = fdgs.make_view(view)
    r.preprocess(cv, sync=True)
    img = r.forward(cv)
    g = ds.zero_grads()
    r.backward(cv, _cuda(dL), g)
    gm = torch.zeros(sc.N, device="cuda")
    train.regularizers(ds, g, lambda_mask=0.01, mask_logit=_cuda(m), mask_eps=eps, grad_mask_logit=gm)
    torch.cuda.synchronize()
    # --- oracle on the kept subset
    sub = sc.subset(np.nonzero(keep)[0])
    o = run_pre(make_oracle(sub), view)
    oimg, _, _, margin = o.forward()
    ok = margin > 1e-4
    assert np.abs(img.cpu().numpy().astype(np.float64) - oimg)[:, ok].max() < 1e-4
    dLm = dL.astype(np.float64) * ok[None]
    g2 = ds.zero_grads()
    r.backward(cv, _cuda(dLm.astype(np.float32)), g2)                       # same threshold-fragile pixels masked on both sides
    gm = torch.zeros(sc.N, device="cuda")
    train.regularizers(ds, g2, lambda_mask=0.01, mask_logit=_cuda(m), mask_eps=eps, grad_mask_logit=gm)
    torch.cuda.synchronize()
    og = o.backward(dLm)
    full_ls, full_lo = np.zeros((sc.N, 4)), np.zeros(sc.N)
    full_ls[keep], full_lo[keep] = og["log_scale"], og["opacity_logit"]
    _, G = T.regularizers(sc.log_scale, sc.quat_l, sc.quat_r, m, 0.0, 0.0, 0.01)
    want = T.mask_backward(m, eps, sc.opacity_logit, full_ls, full_lo) + G["mask_logit"]
    got = gm.cpu().numpy().astype(np.float64)
    err = rel_l2(got, want)
    print("PARITY masked_render grad_mask", err)
    assert err < 1e-3
    # masked primitives: nothing from the render, only the mask loss
    np.testing.assert_allclose(got[~keep], G["mask_logit"][~keep], rtol=1e-5)
    for k in ("mean", "log_scale", "opacity_logit", "sh"):
        assert np.abs(g2[k].cpu().numpy()[~keep]).max() == 0


def test_adam_matches_the_oracle_over_steps_with_a_ragged_count():
    n = 1_000_003
    r = np.random.default_rng(5)
    p0 = r.normal(size=n).astype(np.float32)
    p, m, v = _cuda(p0), torch.zeros(n, device="cuda"), torch.zeros(n, device="cuda")
    op, om, ov = p0.astype(np.float64), np.zeros(n), np.zeros(n)
    # the boundary takes fp32 scalars: both sides get the same fp32-representable hyper-parameters (1 - float32(0.999)
    # differs from 0.001 by 1.3e-5 relative)
    lr, b1, b2, eps = (float(np.float32(x)) for x in (1.6e-3, 0.9, 0.999, 1e-15))
    mag = np.zeros(n)
    for step in range(1, 5):
        g = (r.normal(size=n) * 10.0 ** r.integers(-6, 2, size=n)).astype(np.float32)
        g[r.random(n) < 0.5] = 0.0                                          # most primitives are invisible in a step
        gt = _cuda(g)
        train.adam_step(p, gt, m, v, step, lr, b1, b2, eps, zero_grad=(step % 2 == 0))
        torch.cuda.synchronize()
        mag = np.maximum(mag, np.abs(g.astype(np.float64)))
        op, om, ov = T.adam_step(op, g.astype(np.float64), om, ov, step, lr, b1, b2, eps)
        assert (gt == 0).all().item() == (step % 2 == 0) or not g.any()
        # m = beta1 m + (1 - beta1) g can cancel: the fp32 error is relative to the largest term seen (|m| <= max |g|)
        assert (np.abs(m.cpu().numpy() - om) <= 1e-6 * mag + 1e-30).all()
        assert (np.abs(v.cpu().numpy() - ov) <= 1e-6 * mag * mag + 1e-37).all()
        # a step moves p by at most ~lr: errors are relative to |p| + lr
        assert (np.abs(p.cpu().numpy().astype(np.float64) - op) / (np.abs(op) + lr)).max() < 2e-6 * step
    assert np.abs(op - p0).max() > 1e-3


def test_adam_class_updates_every_array_and_clears_grads():
    sc = scenes.tiny()
    ds = fdgs.DeviceScene.from_scene(sc)
    before = {k: getattr(ds, k).clone() for k in train.PARAMS}
    g = ds.zero_grads()
    for k in train.PARAMS:
        g[k] += 1.0
    opt = train.Adam(ds, {k: 0.01 for k in train.PARAMS})
    opt.step(g)
    torch.cuda.synchronize()
    for k in train.PARAMS:                                                   # first step: p -= lr sign(g)
        np.testing.assert_allclose((before[k] - getattr(ds, k)).cpu().numpy(), 0.01, rtol=1e-4)
        assert g[k].abs().max().item() == 0


@pytest.mark.parametrize("N,L,nt", [(20011, 3, 3), (777, 1, 2), (300, 0, 1)])
def test_decode_compact_matches_the_oracle(N, L, nt):
    c = scenes.compact_model(seed=6, N=N, sh_degree=L, n_time=nt)
    dev = {k: (_cuda(v) if isinstance(v, np.ndarray) else v) for k, v in c.items()}
    ds = train.decode_compact(dev, L, nt)
    torch.cuda.synchronize()
    want = T.decode_compact(c)
    np.testing.assert_array_equal(ds.mean.cpu().numpy().astype(np.float64), want["mean"])        # binary16 -> binary32 is exact
    for k in ("log_scale", "quat_l", "quat_r", "opacity_logit", "sh"):
        got = getattr(ds, k).cpu().numpy().astype(np.float64)
        assert got.shape == want[k].shape
        err = np.abs(got - want[k]).max() / (1.0 + np.abs(want[k]).max())
        print("PARITY decode", N, k, err)
        assert err < 2e-6, k
    # the decoded model is a valid scene for the renderer
    view = scenes.multiview_video(N=8, n_views=1).views[0]
    r = fdgs.Renderer(ds, 320, 240, 1 << 20)
    v2 = scenes.View(view.view, 280.0, 280.0, 160.0, 120.0, 320, 240, 5.0, 10.0, (0, 0, 0))
    D, nvis = r.preprocess(fdgs.make_view(v2), sync=True)
    assert nvis > 0 and D >= nvis


def test_training_loop_through_the_library_recovers_a_perturbed_scene():
    """End to end: fdgs_step_batch (2 views) -> fdgs_regularizers -> fdgs_adam_step on every array, 80 steps.  The targets
    are renders of the unperturbed scene, so the L1 loss must fall well below its start; every array moves, stays finite."""
    sc = scenes.tiny()
    v0 = sc.views[0]
    views = [v0, scenes.View(v0.view, v0.fx, v0.fy, v0.cx, v0.cy, v0.width, v0.height, 0.3, v0.period_T, v0.bg)]
    cvs = [fdgs.make_view(v) for v in views]
    truth = fdgs.DeviceScene.from_scene(sc)
    targets = []
    rt = fdgs.Renderer(truth, v0.width, v0.height, 1 << 16)
    for cv in cvs:
        rt.preprocess(cv)
        targets.append(rt.forward(cv).clone())
    pert = sc.subset(list(range(sc.N)))
    pert.mean[:, :3] += (0.03 * scenes.normal(31, 1, sc.N * 3)).reshape(sc.N, 3).astype(np.float32)
    pert.sh[:, 0, :] += (0.2 * scenes.normal(31, 2, sc.N * 3)).reshape(sc.N, 3).astype(np.float32)
    pert.opacity_logit += (0.5 * scenes.normal(31, 3, sc.N)).astype(np.float32)
    ds = fdgs.DeviceScene.from_scene(pert)
    start = {k: getattr(ds, k).clone() for k in train.PARAMS}
    bs = fdgs.BatchStep(ds, v0.width, v0.height, 1 << 16, 2)
    for r, t in zip(bs.renderers, targets):
        r.target_dev.copy_(t)
    opt = train.Adam(ds, dict(mean=2e-3, log_scale=2e-3, quat_l=1e-3, quat_r=1e-3, opacity_logit=2e-2, sh=5e-3))
    g = ds.zero_grads()
    losses = []
    for it in range(80):
        bs.loss.zero_()
        bs.step(cvs, g)
        train.regularizers(ds, g, lambda_sparse=1e-6, lambda_covt=1e-6)
        opt.step(g, zero_grad=True)
        losses.append(float(bs.loss.sum().item()))
    print("PARITY train_loop loss", losses[0], "->", losses[-1])
    assert losses[-1] < 0.5 * losses[0]
    for k in train.PARAMS:
        p = getattr(ds, k)
        assert torch.isfinite(p).all().item() and (p - start[k]).abs().max().item() > 0
        assert g[k].abs().max().item() == 0                                  # cleared by the optimiser for the next step


def test_regularizers_and_adam_survive_extreme_parameters():
    """Huge / tiny scales, saturated logits, denormal gradients, counts below one vector: finite results that match the oracle."""
    N = 8
    ls = np.array([[-40, -40, -40, -40], [30, 30, 30, 30], [0, 0, 0, 44.5], [-3, -2, -1, 0], [5, -5, 5, -5], [0, 0, 0, -20],
                   [1, 1, 1, 1], [-1, -1, -1, 3]], dtype=np.float32)
    r = np.random.default_rng(3)
    ql = r.normal(size=(N, 4)).astype(np.float32)
    qr = r.normal(size=(N, 4)).astype(np.float32)
    ql[6] *= 1e-18
    qr[7] *= 1e15
    sc = scenes.Scene("x", 0, 1, np.zeros((N, 4), np.float32), ls, ql, qr, np.array([-60, 60, 0, 1, -1, 30, -30, 2], np.float32),
                      np.zeros((N, 1, 3), np.float32), [], 0)
    ds = fdgs.DeviceScene.from_scene(sc)
    g = ds.zero_grads()
    g["log_scale"] += 1e-3
    g["opacity_logit"] += 1e-3
    m = np.array([-50, 50, 0, 1, -1, 20, -20, 0.5], np.float32)
    gm, losses = torch.zeros(N, device="cuda"), torch.zeros(3, device="cuda")
    train.regularizers(ds, g, 0.5, 0.5, 0.5, _cuda(m), 0.3, gm, losses)
    torch.cuda.synchronize()
    L, G = T.regularizers(ls, ql, qr, m, 0.5, 0.5, 0.5)
    want_m = G["mask_logit"] + T.mask_backward(m, 0.3, sc.opacity_logit, np.full((N, 4), 1e-3), np.full(N, 1e-3))
    for k in ("log_scale", "quat_l", "quat_r"):
        got = g[k].cpu().numpy().astype(np.float64) - (1e-3 if k == "log_scale" else 0.0)
        assert np.isfinite(got).all()
        assert np.abs(got - G[k]).max() <= 2e-5 * max(np.abs(G[k]).max(), 1e-30) + 1e-9, k      # fp32 against the largest entry
    got_m = gm.cpu().numpy().astype(np.float64)
    fin = np.isfinite(want_m)                                                # alpha = 1 in fp32 only: 1/(1-alpha) overflows there
    assert np.isfinite(got_m).all() and np.abs(got_m[fin] - want_m[fin]).max() <= 1e-4 * np.abs(want_m[fin]).max()
    np.testing.assert_allclose(losses.cpu().numpy(), [L["sparse"], L["covt"], L["mask"]], rtol=2e-5)
    # Adam on 1, 3 and 5 elements (below / across one 128-bit vector), with a denormal and a huge gradient
    for n in (1, 3, 5):
        p0 = np.linspace(-1, 1, n).astype(np.float32)
        gr = np.array([1e-40, 3e30, -2.0, 0.0, 7e-12][:n], dtype=np.float32)
        p, mm, vv = _cuda(p0), torch.zeros(n, device="cuda"), torch.zeros(n, device="cuda")
        train.adam_step(p, _cuda(gr), mm, vv, 1, float(np.float32(0.01)), float(np.float32(0.9)), float(np.float32(0.999)), float(np.float32(1e-15)))
        torch.cuda.synchronize()
        op, om, ov = T.adam_step(p0.astype(np.float64), gr.astype(np.float64), np.zeros(n), np.zeros(n), 1, float(np.float32(0.01)),
                                 float(np.float32(0.9)), float(np.float32(0.999)), float(np.float32(1e-15)))
        got = p.cpu().numpy().astype(np.float64)
        big = np.abs(gr) > 1e19                                              # g^2 overflows fp32: v = inf, the update is 0 instead of lr
        assert np.isfinite(got).all()
        small = np.abs(gr) < 1e-30                                           # g^2 underflows fp32: m / (0 + eps) instead of sign(g) lr
        sel = ~big & ~small
        np.testing.assert_allclose(got[sel], op[sel], rtol=0, atol=3e-6)


def test_train_entry_points_validate_arguments():
    lib = fdgs.load()
    assert lib.fdgs_mask_apply(None, 0.5, None, None, 10, None) == fdgs.ERR_INVALID
    assert lib.fdgs_mask_apply(None, 0.5, None, None, 0, None) == fdgs.OK
    assert lib.fdgs_adam_step(None, None, None, None, 0, None, 0, None) == fdgs.ERR_INVALID
    x = torch.zeros(16, device="cuda")
    cfg = fdgs.CAdamConfig(0.1, 0.9, 0.999, 1e-15, 0)                        # step 0 is invalid
    import ctypes as C
    assert lib.fdgs_adam_step(x.data_ptr(), x.data_ptr(), x.data_ptr(), x.data_ptr(), 16, C.byref(cfg), 0, None) == fdgs.ERR_INVALID
    cfg.step = 1
    assert lib.fdgs_adam_step(x.data_ptr() + 4, x.data_ptr(), x.data_ptr(), x.data_ptr(), 8, C.byref(cfg), 0, None) == fdgs.ERR_INVALID
    assert lib.fdgs_decode_compact(None, None, None) == fdgs.ERR_INVALID
    ds = fdgs.DeviceScene.from_scene(scenes.tiny())
    with pytest.raises(fdgs.FdgsError):                                      # mask given without a gradient buffer
        train.regularizers(ds, ds.zero_grads(), mask_logit=torch.zeros(ds.N, device="cuda"))
