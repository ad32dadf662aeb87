"""Pins of the oracle's auxiliary channels: rendered depth D = sum_k z_k alpha_k T_k (PAPER.md:L256,
eq. 29 "rendered depth") and accumulated opacity O_gs = 1 - T_final (L233, eq. 25), forward and backward."""
import numpy as np
import pytest

import oracle
from helpers import hand_scene, oracle_for, rel_l2
from paper_2412_20720_b200 import scenes

PARAMS = ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")


def test_single_splat_depth_is_z_times_alpha_and_opacity_is_alpha():
    # isotropic splat on the optical axis at camera depth 4 + 1 = 5 (camera at z = -4, splat at z = +1)
    sc = hand_scene([(0, 0, 1.0, 0.5)], [[-1.0] * 4], logit=[0.3])
    o = oracle_for(sc)
    img, fT, nc, _ = o.forward()
    P = o.prims()
    D = o.depth_map()
    alpha = 1.0 - fT                               # one splat: O = alpha
    assert abs(P.p_cam[0, 2] - 5.0) < 1e-12
    np.testing.assert_allclose(D, 5.0 * alpha, rtol=0, atol=1e-13)
    assert D.max() > 1.0 and alpha.max() < 0.99


def test_two_layer_depth_is_the_over_composite_of_depths():
    # two concentric splats at depths 4.5 and 6: D = z1 a1 + z2 a2 (1 - a1), O = a1 + a2 (1 - a1)
    sc = hand_scene([(0, 0, 0.5, 0.5), (0, 0, 2.0, 0.5)], [[-0.5] * 4, [-0.3] * 4], logit=[-0.5, 0.8])
    o = oracle_for(sc, cfg=dict(oracle.PURE_CFG))
    img, fT, nc, _ = o.forward()
    D = o.depth_map()
    singles = []
    for i in range(2):
        oi = oracle_for(sc.subset([i]), cfg=dict(oracle.PURE_CFG))
        _, fTi, _, _ = oi.forward()
        singles.append(1.0 - fTi)
    a1, a2 = singles
    np.testing.assert_allclose(D, 4.5 * a1 + 6.0 * a2 * (1 - a1), atol=1e-12)
    np.testing.assert_allclose(1 - fT, a1 + a2 * (1 - a1), atol=1e-12)


def test_depth_does_not_change_colour_path():
    sc = scenes.tiny()
    o = oracle_for(sc)
    o.forward()
    G = scenes.upstream_normal(0, 64, 64).astype(np.float64)
    g0 = o.backward(G)
    g1 = o.backward(G, dL_ddepth=np.zeros((64, 64)), dL_dopacity=np.zeros((64, 64)))
    for k in PARAMS:
        np.testing.assert_allclose(g0[k], g1[k], rtol=1e-11, atol=1e-13)     # OpenMP atomics: summation order varies
    assert np.abs(g1["gz"]).max() == 0


def _loss(sc, G, GD, GO, cfg):
    o = oracle_for(sc, cfg=cfg)
    img, fT, nc, mg = o.forward()
    return float((img * G).sum() + (o.depth_map() * GD).sum() + ((1 - fT) * GO).sum()), o, nc, mg


@pytest.mark.parametrize("mode", ["default", "pure"])
def test_aux_backward_matches_central_differences(mode):
    cfg = dict(oracle.DEFAULT_CFG) if mode == "default" else dict(oracle.PURE_CFG)
    for seed in range(100, 120):
        sc = scenes.fd_scene(seed, 6)
        for k in PARAMS:
            setattr(sc, k, getattr(sc, k).astype(np.float64))
        G = 0.3 * scenes.upstream_normal(seed, 64, 64).astype(np.float64)
        GD = scenes.normal(seed, 210, 64 * 64).reshape(64, 64)
        GO = scenes.normal(seed, 211, 64 * 64).reshape(64, 64)
        L0, o0, nc0, mg0 = _loss(sc, G, GD, GO, cfg)
        p0 = o0.prims()
        if not (p0.status == 0).all():
            continue
        if not cfg.get("full_support") and (mg0.min() < 1e-4 or p0.fragility.min() < 1e-4):
            continue
        grads = o0.backward(G, GD, GO)
        lists0 = o0.tile_lists()
        for name in PARAMS:
            arr = getattr(sc, name)
            fd = np.zeros_like(arr)
            it = np.nditer(arr, flags=["multi_index"])
            for x in it:
                idx = it.multi_index
                x0 = float(x)
                h = 1e-6 * max(1.0, abs(x0))
                vals = []
                for sgn in (+1, -1):
                    arr[idx] = x0 + sgn * h
                    Lp, op, ncp, _ = _loss(sc, G, GD, GO, cfg)
                    assert np.array_equal(ncp, nc0) and np.array_equal(op.tile_lists()[1], lists0[1])
                    assert np.array_equal(op.prims().clamp_bits, p0.clamp_bits)
                    vals.append(Lp)
                arr[idx] = x0
                fd[idx] = (vals[0] - vals[1]) / (2 * h)
            assert rel_l2(grads[name], fd) < 1e-5, (name, rel_l2(grads[name], fd))
        # a depth-only loss must reach the parameters only through geometry and opacity, never through colour
        g_depth_only = o0.backward(np.zeros_like(G), GD, None)
        assert np.abs(g_depth_only["sh"]).max() == 0 and np.abs(g_depth_only["mean"]).max() > 0
        return
    pytest.fail("no finite-difference scene far from every threshold found")


def test_densification_indicators_are_norms_of_the_per_view_gradients():
    """spatial position gradient magnitude plus the mu_t gradient as density-control indicators.  Pinned by
    their definition from quantities that are themselves pinned by finite differences: per view |dL/d(u,v)| and |dL/dmu_t|,
    summed over views, with the visibility count."""
    sc = scenes.multiview_video(N=300, width=96, height=64, n_views=3)
    acc = np.zeros((sc.N, 3))
    expect = np.zeros((sc.N, 3))
    for vi in range(3):
        o = oracle_for(sc, vi)
        o.forward()
        G = scenes.upstream_normal(vi, 96, 64).astype(np.float64)
        g = o.backward(G, densify=acc)
        vis = o.prims().status == 0
        expect[:, 0] += np.where(vis, np.linalg.norm(g["mean2d"], axis=1), 0.0)
        expect[:, 1] += np.where(vis, np.abs(g["mean"][:, 3]), 0.0)
        expect[:, 2] += vis
    np.testing.assert_allclose(acc, expect, rtol=1e-12, atol=1e-15)
    assert acc[:, 2].max() == 3 and acc[:, 2].min() == 0 and acc[:, 0].max() > 0 and acc[:, 1].max() > 0
