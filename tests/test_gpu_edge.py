"""GPU edge cases through the C ABI: empty / all-culled scenes, a single tile, depth ties, pair overflow,
gradient accumulation over a batch of views, argument validation."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from helpers import hand_scene, oracle_for
from paper_2412_20720_b200 import scenes


def _f32(sc):
    for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh"):
        setattr(sc, k, np.ascontiguousarray(getattr(sc, k), dtype=np.float32))
    sc.views[0] = sc.views[0].as_fp32()
    return sc


def test_empty_scene_renders_background():
    import gpu_helpers as gh
    sc = _f32(hand_scene(np.zeros((0, 4)), np.zeros((0, 4)), quat_l=np.zeros((0, 4)), quat_r=np.zeros((0, 4)),
                         logit=np.zeros(0), sh=np.zeros((0, 1, 3)), bg=(0.2, 0.4, 0.6), width=70, height=50))
    out = gh.gpu_run(sc, sc.views[0], dL=np.ones((3, 50, 70)))
    assert out["num_pairs"] == 0 and out["num_visible"] == 0
    np.testing.assert_allclose(out["image"], np.array([0.2, 0.4, 0.6])[:, None, None] * np.ones((3, 50, 70)), atol=1e-7)
    assert (out["final_T"] == 1).all() and (out["n_contrib"] == 0).all()


def test_all_culled_and_nonfinite_never_poison():
    import gpu_helpers as gh
    sc = _f32(hand_scene([(0, 0, -10, 0.5), (0, 0, 0, 0.5), (0, 0, 0, 0.5), (0, 0, 0, 9.0)],
                         [[-2] * 4, [np.nan, -2, -2, -2], [-2] * 4, [-2] * 4],
                         quat_l=[[1, 0, 0, 0], [1, 0, 0, 0], [0, 0, 0, 0], [1, 0, 0, 0]], quat_r=[[1, 0, 0, 0]] * 4))
    out = gh.gpu_run(sc, sc.views[0], dL=np.ones((3, 64, 64)))
    assert out["num_visible"] == 0 and out["image"].max() == 0 and np.isfinite(out["image"]).all()
    for k, g in out["grads"].items():
        assert g is None or np.abs(g).max() == 0


def test_single_tile_and_depth_ties():
    import gpu_helpers as gh
    # 16x16 image = one tile (zero tile-id bits); three identical splats: ties resolved by primitive id
    sc = _f32(hand_scene([(0, 0, 0, 0.5)] * 3 + [(0.01, 0, -1.0, 0.5)], [np.log([0.05] * 3 + [1.0])] * 4, logit=[0.5, 0.2, -0.3, 0.1],
                         sh=[[[1, 0, 0]], [[0, 1, 0]], [[0, 0, 1]], [[1, 1, 1]]], width=16, height=16))
    out = gh.gpu_run(sc, sc.views[0])
    o = oracle_for(sc)
    off, ids = o.tile_lists()
    assert list(out["sorted_vals"]) == list(ids) == [3, 0, 1, 2]
    assert np.abs(out["image"] - o.forward()[0]).max() < 1e-5


@pytest.mark.parametrize("far", [40.0, 60000.0])
def test_depth_sort_pass_count_follows_the_depth_range(far):
    """The depth sort runs three 9-bit passes over (fp32 depth bits - bits of znear) and a fourth only if a key has
    bits above the 27th, i.e. a survivor deeper than 2^16 znear: splats from 0.3 to 40 units in front of the camera
    take three passes, splats out to 60 000 units (18 octaves) all four.  Either way the per-tile order is that of the
    oracle's sort on the full depth bits."""
    import gpu_helpers as gh
    rng = np.random.default_rng(11)
    n = 600
    z = np.exp(rng.uniform(np.log(0.3), np.log(far), n))                # log-uniform depth in front of the camera
    xy = rng.uniform(-0.25, 0.25, (n, 2)) * z[:, None]                  # inside the 50 degree frustum at every depth
    mean = np.column_stack([xy, z - 4.0, np.full(n, 0.5)])              # hand_scene puts the camera at z = -4
    ls = np.column_stack([np.log(0.02 * z)] * 3 + [np.zeros(n)])        # footprints of a few pixels at every depth
    sc = _f32(hand_scene(mean, ls, logit=rng.normal(0, 1, n), sh=rng.uniform(0, 2, (n, 1, 3)), width=96, height=80))
    out = gh.gpu_run(sc, sc.views[0])
    from paper_2412_20720_b200 import fdgs
    o = oracle_for(sc)
    P = o.prims()
    off, ids = o.tile_lists()
    assert out["num_visible"] > 0.9 * n
    zs = P.p_cam[P.status == 0, 2]
    assert (zs.max() > 0.2 * 2 ** 16) == (far > 1e4)                    # the case really is on the side of the limit it claims
    order = out["renderer"].export(fdgs.EXPORT_DEPTH_ORDER).cpu().numpy()
    d32 = out["records"][order, 9]
    assert (np.diff(d32) >= 0).all()                                    # survivors in non-decreasing fp32 depth
    same = d32[1:] == d32[:-1]
    assert (order[1:][same] > order[:-1][same]).all()                   # ties in id order
    rep = {}
    frag = P.fragility < gh.FRAG_TOL
    bad = gh.compare_tile_lists(out, P, off, ids, frag, rep)
    assert bad.sum() <= 2, rep
    assert np.abs(out["image"] - o.forward()[0]).max() < 1e-4


def test_pair_overflow_is_reported_and_draws_nothing():
    import gpu_helpers as gh
    from paper_2412_20720_b200 import fdgs
    sc = scenes.tiny()
    with pytest.raises(fdgs.FdgsError) as e:
        gh.gpu_run(sc, sc.views[0], pair_capacity=100)
    assert e.value.code == fdgs.ERR_PAIR_OVERFLOW
    # without the synchronising out-pointers the call sequence still completes and draws only the background
    import torch
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, 64, 64, 100)
    cv = fdgs.make_view(sc.views[0])
    r.preprocess(cv)
    img = r.forward(cv)
    torch.cuda.synchronize()
    assert float(img.abs().max()) == 0.0
    st = r.export(fdgs.EXPORT_STATUS)
    assert st["overflow"] == 1 and st["num_pairs"] == 371


def test_pair_overflow_is_loud_on_every_training_path():
    """a scene that outgrows pair_capacity must not train on a background image with zero gradients in silence.
    fdgs_step_host and fdgs_step_batch (with loss_host) return FDGS_ERR_PAIR_OVERFLOW after their synchronisation, the
    asynchronous fdgs_step_batch writes NaN into the view's loss, and the autograd front end raises."""
    import numpy as np
    import torch
    from paper_2412_20720_b200 import autograd, fdgs
    sc = scenes.tiny()
    v = sc.views[0]
    ds = fdgs.DeviceScene.from_scene(sc)
    cv = fdgs.make_view(v)
    tgt = torch.from_numpy(scenes.target_image(0, 0, 64, 64)).pin_memory()
    r = fdgs.Renderer(ds, 64, 64, 100)
    res = torch.zeros(1).pin_memory()
    with pytest.raises(fdgs.FdgsError) as e:
        r.step_host(cv, tgt, res, ds.zero_grads())
    assert e.value.code == fdgs.ERR_PAIR_OVERFLOW
    bs = fdgs.BatchStep(ds, 64, 64, 100, 2)
    lh = torch.zeros(2).pin_memory()
    with pytest.raises(fdgs.FdgsError) as e:
        bs.step([cv, cv], ds.zero_grads(), targets_host=[tgt, tgt], loss_host=lh, zero_grads=True)
    assert e.value.code == fdgs.ERR_PAIR_OVERFLOW
    for rr in bs.renderers:
        rr.target_dev.copy_(tgt)
    bs.step([cv, cv], ds.zero_grads(), zero_grads=True)          # fully asynchronous: the loss words carry the signal
    torch.cuda.synchronize()
    assert bool(torch.isnan(bs.loss).all())
    # enough capacity: finite losses again on the same objects' code path
    bs2 = fdgs.BatchStep(ds, 64, 64, 4096, 2)
    for rr in bs2.renderers:
        rr.target_dev.copy_(tgt)
    bs2.step([cv, cv], ds.zero_grads(), zero_grads=True)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(bs2.loss).all()) and float(bs2.loss.min()) > 0
    rast = autograd.Rasterizer(sc.sh_degree, sc.n_time, 64, 64, 100)
    params = {k: getattr(ds, k).clone().requires_grad_(True) for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")}
    with pytest.raises(fdgs.FdgsError) as e:
        rast(params, cv)
    assert e.value.code == fdgs.ERR_PAIR_OVERFLOW


def test_batch_of_views_accumulates():
    """Gradient buffers are accumulated into: sum over views of grads == grads of the summed loss (L324 batch)."""
    import gpu_helpers as gh
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=5000, width=128, height=96, n_views=3)
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, 128, 96, 1 << 20)
    total = ds.zero_grads()
    singles = []
    for vi, v in enumerate(sc.views):
        cv = fdgs.make_view(v)
        dL = torch.from_numpy(scenes.upstream_normal(vi, 128, 96)).cuda()
        g1 = ds.zero_grads()
        for g in (g1, total):
            r.preprocess(cv); r.forward(cv); r.backward(cv, dL, g)
        singles.append(g1)
    torch.cuda.synchronize()
    for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh"):
        s = sum(g[k].double() for g in singles)
        assert gh.rel_l2(total[k].cpu().numpy(), s.cpu().numpy()) < 1e-5
        assert float(total[k].abs().max()) > 0


def test_argument_validation():
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.tiny()
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, 64, 64, 4096)
    cv = fdgs.make_view(sc.views[0])
    ds.sh_degree = 7
    r._cs = ds.c_struct()
    with pytest.raises(fdgs.FdgsError) as e:
        r.preprocess(cv)
    assert e.value.code == fdgs.ERR_INVALID
    ds.sh_degree = 1
    r._cs = ds.c_struct()
    r.ws_bytes = 1024
    with pytest.raises(fdgs.FdgsError) as e:
        r.preprocess(cv)
    assert e.value.code == fdgs.ERR_WORKSPACE
    # thresholds that do not describe a renderer are rejected, not rendered with (alpha_max >= 1 with
    # transmittance_min = 0 divides by zero in the backward; a non-positive guard, cutoff or near plane, a negative dilation)
    r = fdgs.Renderer(ds, 64, 64, 4096)
    for bad in (dict(alpha_min=0.5, alpha_max=0.25), dict(alpha_max=1.5), dict(alpha_min=-0.1), dict(transmittance_min=1.0),
                dict(transmittance_min=-1e-3), dict(dilation=-0.3), dict(cutoff_sigma=0.0), dict(guard=0.0), dict(znear=0.0),
                dict(marginal_min=-0.05), dict(marginal_min=float("nan")), dict(alpha_max=float("nan"))):
        r.cfg = fdgs.default_config(**bad)
        with pytest.raises(fdgs.FdgsError) as e:
            r.preprocess(cv)
        assert e.value.code == fdgs.ERR_INVALID, bad
    r.cfg = fdgs.default_config()
    r.preprocess(cv); r.forward(cv)
    # misaligned arrays that the kernels read with 128-bit accesses: an offset view of the 4DSH gradient, of the features
    g = ds.zero_grads()
    big = torch.zeros(g["sh"].numel() + 1, device="cuda")
    g_bad = dict(g, sh=big[1:].view_as(g["sh"]))
    with pytest.raises(fdgs.FdgsError) as e:
        r.backward(cv, torch.zeros(3, 64, 64, device="cuda"), g_bad)
    assert e.value.code == fdgs.ERR_INVALID
    feat_big = torch.zeros(ds.N * 4 + 1, device="cuda")
    with pytest.raises(fdgs.FdgsError) as e:
        r.features_forward(cv, feat_big[1:].view(ds.N, 4))
    assert e.value.code == fdgs.ERR_INVALID
    torch.cuda.synchronize()


def test_step_host_matches_device_path():
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=5000, width=128, height=96, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, 128, 96, 1 << 20)
    cv = fdgs.make_view(sc.views[0])
    tgt = torch.from_numpy(scenes.target_image(3, 0, 128, 96)).pin_memory()
    res = torch.zeros(1).pin_memory()
    g = ds.zero_grads()
    r.step_host(cv, tgt, res, g)
    img = r.image.clone()
    loss_ref = float((img.double().cpu() - tgt.double()).abs().mean())
    assert abs(float(res[0]) - loss_ref) < 1e-5 * max(1.0, loss_ref)
    g2 = ds.zero_grads()
    r.preprocess(cv); r.forward(cv)
    r.loss.zero_(); r.l1_loss(tgt.cuda()); r.backward(cv, r.dL_dimage, g2)
    torch.cuda.synchronize()
    assert torch.allclose(g["sh"], g2["sh"], rtol=1e-4, atol=1e-9)
    out = torch.zeros(3 * 96 * 128).pin_memory()
    r.step_host(cv, None, out, None)
    assert torch.equal(out.view(3, 96, 128), r.image.cpu())


def test_step_batch_matches_view_by_view():
    """fdgs_step_batch (views on concurrent worker streams, chained gradient accumulation) == the three calls view by view."""
    import gpu_helpers as gh
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=20000, width=200, height=150, n_views=4)
    ds = fdgs.DeviceScene.from_scene(sc)
    cvs = [fdgs.make_view(v) for v in sc.views]
    tg = [torch.from_numpy(scenes.target_image(sc.seed, i, 200, 150)) for i in range(4)]
    # reference: sequential, one renderer
    r = fdgs.Renderer(ds, 200, 150, 1 << 21)
    g_ref = ds.zero_grads()
    losses_ref = []
    for cv, t in zip(cvs, tg):
        r.loss.zero_()
        r.preprocess(cv); r.forward(cv); r.l1_loss(t.cuda()); r.backward(cv, r.dL_dimage, g_ref)
        losses_ref.append(float(r.loss[0]))
    torch.cuda.synchronize()
    # batched, host targets, losses read back
    bs = fdgs.BatchStep(ds, 200, 150, 1 << 21, 4)
    g = ds.zero_grads()
    loss_host = torch.zeros(4).pin_memory()
    for _ in range(3):     # repeated calls reuse the worker streams and events
        for v in g.values():
            if v is not None:
                v.zero_()
        bs.step(cvs, g, targets_host=[t.pin_memory() for t in tg], loss_host=loss_host)
    for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh"):
        assert gh.rel_l2(g[k].cpu().numpy(), g_ref[k].cpu().numpy()) < 1e-5, k
    assert np.allclose(loss_host.numpy(), np.array(losses_ref), rtol=1e-5)
    # device-resident targets, asynchronous, gradients zeroed by the library (they start from garbage here)
    g2 = {k: (torch.full_like(v, 7.0) if v is not None else None) for k, v in ds.zero_grads().items()}
    bs.step(cvs, g2, zero_grads=True)
    torch.cuda.synchronize()
    assert gh.rel_l2(g2["sh"].cpu().numpy(), g_ref["sh"].cpu().numpy()) < 1e-5
    with pytest.raises(ValueError):
        fdgs.BatchStep(ds, 200, 150, 1 << 21, 9)


@pytest.mark.parametrize("n_views,sh_degree,n_time", [(2, 3, 1), (3, 3, 2), (4, 3, 3), (4, 3, 4),      # one colour pass for the batch
                                                       (5, 3, 3), (3, 2, 3), (2, 3, 5)])                # per-view chain
def test_step_batch_backward_preprocess_variants(n_views, sh_degree, n_time):
    """The backward preprocess of fdgs_step_batch — one colour pass over the union of the views' survivors where the scene
    allows it (sh_degree 3, <= 4 Fourier orders, <= 4 views), the per-view chain otherwise — adds to the caller's arrays
    exactly what the view-by-view calls add, with and without FDGS_STEP_ZERO_GRADS."""
    import gpu_helpers as gh
    import torch
    from paper_2412_20720_b200 import fdgs
    W, H, N = 136, 104, 6000
    base = scenes.multiview_video(N=N, width=W, height=H, n_views=n_views)
    K = n_time * (sh_degree + 1) ** 2
    sh = np.ascontiguousarray(np.resize(base.sh.reshape(N, -1), (N, 3 * K)).reshape(N, K, 3))
    sc = scenes.Scene("variant", sh_degree, n_time, base.mean, base.log_scale, base.quat_l, base.quat_r, base.opacity_logit, sh,
                      base.views, base.seed)
    ds = fdgs.DeviceScene.from_scene(sc)
    cvs = [fdgs.make_view(v) for v in sc.views]
    tg = [torch.from_numpy(scenes.target_image(sc.seed, i, W, H)).cuda() for i in range(n_views)]
    keys = ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")
    r = fdgs.Renderer(ds, W, H, 1 << 20)
    g_ref = ds.zero_grads()
    seen = 0
    for cv, t in zip(cvs, tg):
        r.loss.zero_()
        D, nvis = r.preprocess(cv, sync=True); r.forward(cv); r.l1_loss(t); r.backward(cv, r.dL_dimage, g_ref)
        seen += nvis
    torch.cuda.synchronize()
    assert seen > 1000
    ref = {k: g_ref[k].cpu().numpy().astype(np.float64) for k in keys}
    bs = fdgs.BatchStep(ds, W, H, 1 << 20, n_views)
    for rr, t in zip(bs.renderers, tg):
        rr.target_dev.copy_(t)
    g = ds.zero_grads()
    for rep in (1, 2):                                           # the second call adds to what the first one left
        bs.step(cvs, g)
        torch.cuda.synchronize()
        for k in keys:
            assert gh.rel_l2(g[k].cpu().numpy(), rep * ref[k]) < 1e-5, (k, rep)
    bs.step(cvs, g, zero_grads=True)                             # cleared by the library, then written
    torch.cuda.synchronize()
    for k in keys:
        assert gh.rel_l2(g[k].cpu().numpy(), ref[k]) < 1e-5, k


def test_autograd_front_end_matches_the_c_abi_path():
    """paper_2412_20720_b200.autograd.Rasterizer: loss.backward() == fdgs_render_backward(_aux) with the same upstream."""
    import gpu_helpers as gh
    import torch
    from paper_2412_20720_b200 import autograd, fdgs
    sc = scenes.multiview_video(N=8000, width=160, height=112, n_views=1)
    view = sc.views[0]
    ds = fdgs.DeviceScene.from_scene(sc)
    params = {k: getattr(ds, k).clone().requires_grad_(True) for k in autograd.PARAM_KEYS}
    rast = autograd.Rasterizer(sc.sh_degree, sc.n_time, 160, 112, 1 << 20)
    tgt = torch.from_numpy(scenes.target_image(3, 0, 160, 112)).cuda()
    # colour only
    img = rast(params, view)
    (img - tgt).abs().mean().backward()
    r = fdgs.Renderer(ds, 160, 112, 1 << 20)
    cv = fdgs.make_view(view)
    g = ds.zero_grads()
    r.preprocess(cv); r.forward(cv); r.loss.zero_(); r.l1_loss(tgt); r.backward(cv, r.dL_dimage, g)
    torch.cuda.synchronize()
    assert torch.equal(img.detach(), r.image)
    for k in autograd.PARAM_KEYS:
        assert gh.rel_l2(params[k].grad.cpu().numpy(), g[k].cpu().numpy()) < 1e-5, k
        params[k].grad = None
    # colour + depth + opacity
    img, depth, opac = rast(params, view, aux=True)
    loss = (img * img).sum() * 1e-4 + (depth * 0.01).sum() + (opac * opac).sum() * 1e-3
    loss.backward()
    g2 = ds.zero_grads()
    r.preprocess(cv); r.forward_aux(cv)
    r.backward_aux(cv, (2e-4 * r.image).contiguous(), torch.full_like(r.depth_map, 0.01), (2e-3 * (1 - r.final_T)).contiguous(), g2)
    torch.cuda.synchronize()
    for k in autograd.PARAM_KEYS:
        assert gh.rel_l2(params[k].grad.cpu().numpy(), g2[k].cpu().numpy()) < 1e-5, k
    # a stale graph is refused instead of silently using the wrong workspace state
    a = rast(params, view)
    rast(params, view)
    with pytest.raises(RuntimeError, match="rendered again"):
        a.sum().backward()


def test_densification_indicators_match_the_oracle():
    """grads.densify [N,3]: |dL/d(u,v)|, |dL/dmu_t| and visibility count, accumulated view by view."""
    import gpu_helpers as gh
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=6000, width=160, height=112, n_views=3)
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, 160, 112, 1 << 20)
    g = ds.zero_grads(with_mean2d=True, with_densify=True)
    acc = np.zeros((sc.N, 3))
    fragile = np.zeros(sc.N, dtype=bool)
    for vi, v in enumerate(sc.views):
        o = oracle_for(sc, vi)
        o.forward()
        dL = scenes.upstream_normal(vi, 160, 112)
        o.backward(dL.astype(np.float64), densify=acc)
        fragile |= o.prims().fragility < gh.FRAG_TOL
        cv = fdgs.make_view(v)
        r.preprocess(cv); r.forward(cv); r.backward(cv, torch.from_numpy(dL).cuda(), g)
    torch.cuda.synchronize()
    dn = g["densify"].cpu().numpy().astype(np.float64)
    keep = ~fragile
    assert np.array_equal(dn[keep, 2], acc[keep, 2]) and dn[:, 2].max() == 3
    assert gh.rel_l2(dn[keep, 0], acc[keep, 0]) < 1e-3 and gh.rel_l2(dn[keep, 1], acc[keep, 1]) < 1e-3
    # the batched step accumulates the same indicators
    bs = fdgs.BatchStep(ds, 160, 112, 1 << 20, 3)
    g2 = ds.zero_grads(with_densify=True)
    for i, rr in enumerate(bs.renderers):
        rr.target_dev.copy_(torch.from_numpy(scenes.target_image(3, i, 160, 112)).cuda())
    bs.step([fdgs.make_view(v) for v in sc.views], g2)
    torch.cuda.synchronize()
    assert torch.equal(g2["densify"][:, 2], g["densify"][:, 2]) and float(g2["densify"][:, 1].max()) > 0


def test_whole_step_replays_from_a_cuda_graph():
    """The call sequence issues no host-memory copies and no synchronisation: preprocess + forward + loss + backward is
    captured once into a CUDA graph and replayed with the same result."""
    import gpu_helpers as gh
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=8000, width=160, height=112, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, 160, 112, 1 << 20)
    cv = fdgs.make_view(sc.views[0])
    tgt = torch.from_numpy(scenes.target_image(3, 0, 160, 112)).cuda()
    g_ref = ds.zero_grads()
    r.preprocess(cv); r.forward(cv); r.loss.zero_(); r.l1_loss(tgt); r.backward(cv, r.dL_dimage, g_ref)
    torch.cuda.synchronize()
    img_ref = r.image.clone()
    g = ds.zero_grads()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            r.preprocess(cv); r.forward(cv); r.loss.zero_(); r.l1_loss(tgt); r.backward(cv, r.dL_dimage, g)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(3):
        for v in g.values():
            if v is not None:
                v.zero_()
        r.image.zero_()
        graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(r.image, img_ref)
    for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh"):
        assert gh.rel_l2(g[k].cpu().numpy(), g_ref[k].cpu().numpy()) < 1e-5, k


def test_marginal_filter_off_with_underflowing_weight_gives_finite_zero_gradients():
    """marginal_min = 0 (urban variant): a primitive 60 sigma away in time has o = sigmoid * w = 0 in fp32; it
    is listed, composites nothing, and its gradients are exactly zero (regression: dL/do = S1 / o used to be 0 * inf)."""
    import gpu_helpers as gh
    sc = _f32(hand_scene([(0.0, 0.0, 0.0, 0.5), (0.1, 0.0, 0.5, 30.5)], [[-1.5, -1.5, -1.5, -0.7]] * 2, logit=[0.2, 0.4], sh=np.full((2, 1, 3), 1.0)))
    out = gh.gpu_run(sc, sc.views[0], cfg_overrides=dict(marginal_min=0.0), dL=np.ones((3, 64, 64)))
    assert out["num_visible"] == 2
    for k, g in out["grads"].items():
        if g is not None:
            assert np.isfinite(g).all(), k
    assert np.abs(out["grads"]["mean"][1]).max() == 0 and np.abs(out["grads"]["sh"][1]).max() == 0
    assert np.abs(out["grads"]["mean"][0]).max() > 0
    assert np.isfinite(out["g9"]).all()


def test_default_threshold_instantiations_agree_with_the_generic_kernels():
    """The blend kernels run an instantiation with the thresholds of [23] as immediates when the configuration holds exactly
    those values.  Moving alpha_max by one ulp selects the generic kernels (thresholds read from the
    kernel arguments): image, transmittance, contributor counts and gradients must agree up to the effect of that ulp."""
    import gpu_helpers as gh
    sc = _f32(scenes.tiny(seed=7, N=2000))
    v = sc.views[0]
    rng = np.random.default_rng(11)
    dL = rng.standard_normal((3, v.height, v.width))
    a = gh.gpu_run(sc, v, dL=dL)
    amax = float(np.nextafter(np.float32(0.99), np.float32(0.0)))
    b = gh.gpu_run(sc, v, cfg_overrides=dict(alpha_max=amax), dL=dL)
    assert a["num_pairs"] == b["num_pairs"] and a["num_pairs"] > 0
    assert np.abs(a["image"] - b["image"]).max() <= 1e-6
    assert np.abs(a["final_T"] - b["final_T"]).max() <= 1e-6
    assert (a["n_contrib"] != b["n_contrib"]).mean() <= 1e-3
    for k, g in a["grads"].items():
        if g is None:
            continue
        den = np.linalg.norm(g)
        assert den > 0 or np.linalg.norm(b["grads"][k]) == 0, k
        if den > 0:
            assert np.linalg.norm(g - b["grads"][k]) / den <= 1e-4, k
