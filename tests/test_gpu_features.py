"""GPU parity of the feature channels and of the optical flow (L410) against the float64 oracle,
through the C ABI.  Tolerances as for the colour path: maps max-abs <= 1e-4 over pixels whose alpha / transmittance
tests are not within 1e-4 of a threshold and whose tile lists agree; gradients rel-L2 <= 1e-3."""
import numpy as np
import pytest
import torch

from gpu_helpers import compare_prims, compare_tile_lists, flagged_pixels, rel_l2
from helpers import make_oracle, run_pre
from paper_2412_20720_b200 import fdgs, scenes

pytestmark = pytest.mark.gpu


def _setup(sc, view, cap=1 << 20):
    ds = fdgs.DeviceScene.from_scene(sc)
    r = fdgs.Renderer(ds, view.width, view.height, cap)
    cv = fdgs.make_view(view)
    r.preprocess(cv, sync=True)
    r.forward(cv)
    return ds, r, cv


def _zero_bg(view):
    return scenes.View(view.view, view.fx, view.fy, view.cx, view.cy, view.width, view.height, view.t, view.period_T, (0.0, 0.0, 0.0))


def _flags(r, o, view):
    """Pixels excluded from the strict comparison (protocol of DESIGN.md section 3)."""
    P = o.prims()
    gpu = dict(ranges=r.export(fdgs.EXPORT_RANGES).cpu().numpy(), sorted_vals=r.export(fdgs.EXPORT_SORTED_VALS).cpu().numpy(),
               sorted_keys=r.export(fdgs.EXPORT_SORTED_KEYS).cpu().numpy())
    off, ids = o.tile_lists()
    rep = {}
    bad = compare_tile_lists(gpu, P, off, ids, P.fragility < 1e-5, rep)
    _, _, _, margin = o.forward()
    return flagged_pixels(bad, margin, view.width, view.height)


@pytest.mark.parametrize("name,C", [("tiny", 5), ("object_reduced", 32)])
def test_feature_maps_and_gradients_match_the_oracle(name, C):
    if name == "tiny":
        sc = scenes.tiny()
        view = _zero_bg(sc.views[0])
    else:
        sc = scenes.single_object(N=6000, width=250, height=190)              # ragged tiles, K = 48, D = 32 as in L603
        view = _zero_bg(sc.views[0])
    feat = scenes.normal(21, 3, sc.N * C).reshape(sc.N, C).astype(np.float32)
    G = scenes.normal(22, 4, C * view.width * view.height).reshape(C, view.height, view.width).astype(np.float32)
    ds, r, cv = _setup(sc, view)
    ft = torch.from_numpy(feat).cuda()
    F = r.features_forward(cv, ft)
    torch.cuda.synchronize()
    o = run_pre(make_oracle(sc), view)
    flag = _flags(r, o, view)
    assert flag.mean() < 0.05
    want = o.render_features(feat.astype(np.float64))
    err = np.abs(F.cpu().numpy().astype(np.float64) - want)[:, ~flag].max()
    print("PARITY features", name, C, "max_abs", err, "flagged", float(flag.mean()))
    assert err < 1e-4 * max(1.0, np.abs(want).max())
    # backward with the flagged pixels masked on both sides
    Gm = G.astype(np.float64) * (~flag)[None]
    gf = torch.zeros_like(ft) + 0.5                                           # += semantics
    g = ds.zero_grads()
    r.features_backward(cv, ft, torch.from_numpy(Gm.astype(np.float32)).cuda(), gf, g)
    torch.cuda.synchronize()
    ogf, ogp = o.backward_features(feat.astype(np.float64), Gm)
    e = rel_l2(gf.cpu().numpy().astype(np.float64) - 0.5, ogf)
    print("PARITY features", name, "grad_feat", e)
    assert e < 1e-3
    P = o.prims()
    keep = P.fragility >= 1e-5
    for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit"):
        e = rel_l2(g[k].cpu().numpy().astype(np.float64)[keep], ogp[k][keep])
        print("PARITY features", name, k, e)
        assert e < 1e-3, k
    assert g["sh"].abs().max().item() == 0
    # features only (no parameter gradients requested)
    gf2 = torch.zeros_like(ft)
    r.features_backward(cv, ft, torch.from_numpy(Gm.astype(np.float32)).cuda(), gf2, None)
    torch.cuda.synchronize()
    assert rel_l2(gf2.cpu().numpy(), ogf) < 1e-3


@pytest.mark.parametrize("C", [1, 3, 4, 7, 16, 33, 36, 40, 67])
def test_channel_counts_cover_every_pass_combination(C):
    """32-, 16- and 4-channel forward instantiations, aligned and ragged row slices, one to three backward passes."""
    sc = scenes.tiny()
    view = _zero_bg(sc.views[0])
    feat = scenes.normal(40 + C, 3, sc.N * C).reshape(sc.N, C).astype(np.float32)
    G = scenes.normal(50 + C, 4, C * view.width * view.height).reshape(C, view.height, view.width).astype(np.float32)
    ds, r, cv = _setup(sc, view)
    ft = torch.from_numpy(feat).cuda()
    F = r.features_forward(cv, ft)
    gf = torch.zeros_like(ft)
    r.features_backward(cv, ft, torch.from_numpy(G).cuda(), gf, None)
    torch.cuda.synchronize()
    o = run_pre(make_oracle(sc), view)
    margin = o.forward()[3]
    ok = margin > 1e-4
    want = o.render_features(feat.astype(np.float64))
    assert np.abs(F.cpu().numpy().astype(np.float64) - want)[:, ok].max() < 1e-4
    if ok.all():                                                              # no threshold-fragile pixel in this scene
        ogf, _ = o.backward_features(feat.astype(np.float64), G.astype(np.float64))
        assert rel_l2(gf.cpu().numpy(), ogf) < 1e-3


def test_constant_feature_is_one_minus_final_T_and_colour_path_is_untouched():
    sc = scenes.tiny()
    view = sc.views[0]
    ds, r, cv = _setup(sc, view)
    img0, fT0, nc0 = r.image.clone(), r.final_T.clone(), r.n_contrib.clone()
    F = r.features_forward(cv, torch.ones((sc.N, 1), device="cuda"))
    torch.cuda.synchronize()
    assert (F[0] - (1 - r.final_T)).abs().max().item() < 2e-6
    assert torch.equal(img0, r.image) and torch.equal(fT0, r.final_T) and torch.equal(nc0, r.n_contrib)
    # the colour backward still works on the same workspace afterwards
    g = ds.zero_grads()
    r.backward(cv, torch.from_numpy(scenes.upstream_normal(0, 64, 64)).cuda(), g)
    torch.cuda.synchronize()
    assert g["sh"].abs().max().item() > 0


@pytest.mark.parametrize("name", ["tiny_random", "video_tilted"])
def test_splat_flow_and_rendered_flow_match_the_oracle(name):
    if name == "tiny_random":
        sc = scenes.tiny()
        view, d = _zero_bg(sc.views[0]), 0.04
    else:
        sc = scenes.multiview_video(N=30000, width=320, height=240, n_views=1)
        view, d = _zero_bg(sc.views[0]), 1.0 / 30.0
    ds, r, cv = _setup(sc, view)
    flow = r.splat_flow(cv, d)
    torch.cuda.synchronize()
    o = run_pre(make_oracle(sc), view)
    P = o.prims()
    want = o.splat_flow(view.view, (view.fx, view.fy, view.cx, view.cy), float(np.float32(d)))
    got = flow.cpu().numpy().astype(np.float64)
    vis_g = r.export(fdgs.EXPORT_TILES_TOUCHED).cpu().numpy() > 0
    same = (P.status == 0) == vis_g                                           # fragile cull decisions excluded
    scale = np.abs(want).max()
    err = np.abs(got - want)[same].max() / scale
    print("PARITY flow", name, "max_rel_to_max", err, "max_flow_px", scale)
    assert scale > 0.05 and err < 1e-4
    assert np.abs(got[~vis_g]).max() == 0
    # rendered flow map = features forward with C = 2
    Fm = r.features_forward(cv, flow)
    torch.cuda.synchronize()
    flag = _flags(r, o, view)
    wantm = o.render_features(want)
    e = np.abs(Fm.cpu().numpy().astype(np.float64) - wantm)[:, ~flag].max()
    print("PARITY flow map", name, e)
    assert e < 1e-4 * max(1.0, np.abs(wantm).max())


def test_feature_entry_points_validate_and_handle_empty_scenes():
    sc = scenes.tiny().subset([])
    view = scenes.tiny().views[0]
    ds, r, cv = _setup(sc, view, cap=1 << 10)
    F = r.features_forward(cv, torch.zeros((0, 4), device="cuda"))
    torch.cuda.synchronize()
    assert F.shape == (4, 64, 64) and F.abs().max().item() == 0
    sc2 = scenes.tiny()
    ds2, r2, cv2 = _setup(sc2, sc2.views[0])
    import ctypes as C
    rc = r2.lib.fdgs_render_features_forward(C.byref(r2._cs), C.byref(cv2), C.byref(r2.cfg), r2.ws.data_ptr(), r2.ws_bytes, r2.cap,
                                             None, None, 3, None, 0, None)
    assert rc == fdgs.ERR_INVALID
    with pytest.raises(fdgs.FdgsError):                                       # C = 0 channels
        r2.features_forward(cv2, torch.zeros((sc2.N, 0), device="cuda"))
