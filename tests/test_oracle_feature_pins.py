"""Pins of the oracle's feature channels (eq. 6 "with the color c replaced by the ... feature vector") and of
the rendered optical flow (L410: the projected displacement of mu_xyz|t between two frames, rendered with eq. 6)."""
import numpy as np

import oracle
from helpers import hand_scene, make_oracle, oracle_for, run_pre
from paper_2412_20720_b200 import scenes


def _no_bg(sc):
    v = sc.views[0]
    sc.views[0] = scenes.View(v.view, v.fx, v.fy, v.cx, v.cy, v.width, v.height, v.t, v.period_T, (0.0, 0.0, 0.0))
    return sc


def test_constant_feature_renders_the_accumulated_opacity_and_features_are_linear():
    sc = _no_bg(scenes.tiny())
    o = oracle_for(sc)
    _, fT, _, _ = o.forward()
    r = np.random.default_rng(0)
    f1, f2 = r.normal(size=(sc.N, 5)), r.normal(size=(sc.N, 5))
    F1, F2 = o.render_features(f1), o.render_features(f2)
    ones = o.render_features(np.ones((sc.N, 1)))
    np.testing.assert_allclose(ones[0], 1.0 - fT, atol=1e-13)              # sum_k alpha_k T_k = 1 - T_final (eq. 25's O_gs)
    np.testing.assert_allclose(o.render_features(2.0 * f1 - 0.5 * f2), 2.0 * F1 - 0.5 * F2, atol=1e-12)
    assert F1.shape == (5, 64, 64) and np.abs(F1[4]).max() > 0.01            # 5 channels = two passes, the second ragged


def test_features_equal_to_the_colours_reproduce_the_image():
    sc = _no_bg(scenes.tiny())
    o = oracle_for(sc)
    img = o.forward()[0]
    rgb = np.nan_to_num(o.prims().rgb)                                       # eq. 20 colours of the visible primitives
    np.testing.assert_allclose(o.render_features(rgb), img, atol=1e-14)


def test_single_splat_feature_is_feature_times_alpha():
    sc = hand_scene([(0, 0, 1.0, 0.5)], [[-1.0] * 4], logit=[0.3])
    o = oracle_for(sc)
    _, fT, _, _ = o.forward()
    F = o.render_features(np.array([[0.25, -3.0, 7.0, 1.5]]))
    for c, f in enumerate((0.25, -3.0, 7.0, 1.5)):
        np.testing.assert_allclose(F[c], f * (1.0 - fT), atol=1e-13)


def test_feature_backward_matches_central_differences():
    sc = _no_bg(scenes.fd_scene(3))
    view = sc.views[0]
    cfg = dict(oracle.PURE_CFG)
    C = 4
    r = np.random.default_rng(1)
    feat = r.normal(size=(sc.N, C))
    G = r.normal(size=(C, view.height, view.width))

    def loss(scene, f):
        return float((run_pre(make_oracle(scene), view, cfg).render_features(f) * G).sum())

    o = run_pre(make_oracle(sc), view, cfg)
    gf, gp = o.backward_features(feat, G)
    h = 1e-6
    for idx in [(0, 0), (2, 3), (5, 1), (7, 2)]:
        up, dn = feat.copy(), feat.copy()
        up[idx] += h
        dn[idx] -= h
        fd = (loss(sc, up) - loss(sc, dn)) / (2 * h)
        assert abs(fd - gf[idx]) <= 1e-6 * max(1.0, abs(fd)), (idx, fd, gf[idx])
    for name, idx in [("mean", (1, 0)), ("mean", (4, 3)), ("log_scale", (2, 1)), ("log_scale", (6, 3)), ("quat_l", (3, 2)),
                      ("quat_r", (0, 1)), ("opacity_logit", (5,))]:
        vals = []
        for sgn in (+1, -1):
            s2 = sc.subset(list(range(sc.N)))
            for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit"):
                setattr(s2, k, getattr(s2, k).astype(np.float64))
            getattr(s2, name)[idx] += sgn * h
            vals.append(loss(s2, feat))
        fd = (vals[0] - vals[1]) / (2 * h)
        assert abs(fd - gp[name][idx]) <= 1e-5 * max(1.0, abs(fd)), (name, idx, fd, gp[name][idx])
    assert np.abs(gp["sh"]).max() == 0                                       # the colour coefficients do not enter


def test_flow_is_the_difference_of_the_projections_at_two_times():
    sc = scenes.tiny()
    view = sc.views[0]
    intr = (view.fx, view.fy, view.cx, view.cy)
    d = 0.04
    o0 = oracle_for(sc, cfg=dict(marginal_min=0.0))
    o1 = oracle_for(sc, cfg=dict(marginal_min=0.0), t=view.t + d)
    P0, P1 = o0.prims(), o1.prims()
    flow = o0.splat_flow(view.view, intr, d)
    both = (P0.status == 0) & (P1.status == 0)
    assert both.sum() > 100
    np.testing.assert_allclose(flow[both], P1.uv[both] - P0.uv[both], atol=1e-9)    # full preprocess at t + d, independently
    assert np.abs(flow[both]).max() > 0.5                                     # random 4D rotations: the splats do move
    o2 = oracle_for(sc)                                                       # default thresholds: culled primitives have no flow
    f2, st = o2.splat_flow(view.view, intr, d), o2.prims().status
    assert (st != 0).sum() > 10 and np.abs(f2[st != 0]).max() == 0


def test_flow_vanishes_without_space_time_rotation():
    # q_r = (a, b, c, -d): pure spatial rotation => Sigma_1:3,4 = 0 => mu_xyz|t does not move
    sc = scenes.tiny()
    sc.quat_r[:] = sc.quat_l * np.array([1, 1, 1, -1], dtype=np.float32)
    view = sc.views[0]
    o = oracle_for(sc)
    flow = o.splat_flow(view.view, (view.fx, view.fy, view.cx, view.cy), 0.1)
    assert np.abs(flow).max() < 1e-9
