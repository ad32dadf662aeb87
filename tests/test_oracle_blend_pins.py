"""Pins for the float64 oracle, part 2: tile lists (brute force), the blend loop (closed forms and a
direct numpy evaluation of eq. 6), invariants of the whole renderer, and the analytic backward
against central finite differences (north_star: <= 8 primitives, 1e-5 relative)."""
import numpy as np
import pytest

import oracle
from helpers import hand_scene, make_oracle, oracle_for, rel_l2, run_pre
from paper_2412_20720_b200 import scenes

Y00 = 0.28209479177387814


# ------------------------------------------------------------------ tile lists
def test_tile_lists_bruteforce():
    sc = scenes.tiny()
    o = oracle_for(sc)
    p = o.prims()
    off, ids = o.tile_lists()
    tiles_x = 4
    vis = np.where(p.status == oracle.STATUS_VISIBLE)[0]
    total = 0
    for tl in range(16):
        tx, ty = tl % tiles_x, tl // tiles_x
        members = []
        for i in vis:
            u, v, r = p.uv[i, 0], p.uv[i, 1], p.radius[i]
            # the tile [16tx,16tx+16) x [16ty,16ty+16) lies in the rect floor((u-r)/16) .. ceil((u+r)/16)
            if np.floor((u - r) / 16) <= tx < np.ceil((u + r) / 16) and np.floor((v - r) / 16) <= ty < np.ceil((v + r) / 16):
                members.append(i)
        bits = lambda i: np.float32(p.p_cam[i, 2]).view(np.uint32)
        members.sort(key=lambda i: (int(bits(i)), i))
        got = ids[off[tl]:off[tl + 1]]
        assert list(got) == members
        total += len(members)
    assert total == off[-1] and total > 100


def test_depth_ties_resolved_by_primitive_id():
    # three identical-depth splats in one tile: list order = id order
    sc = hand_scene([(0, 0, 0, 0.5)] * 3, [np.log([0.05] * 3 + [1.0])] * 3)
    off, ids = oracle_for(sc).tile_lists()
    for tl in range(16):
        assert list(ids[off[tl]:off[tl + 1]]) in ([], [0, 1, 2])


# ------------------------------------------------------------------ blend closed forms
def _layers(zs, logits, cols, s=0.5, cfg=None, bg=(0, 0, 0)):
    """Large isotropic splats stacked on the optical axis; colour via DC only."""
    n = len(zs)
    sh = np.array([[(np.array(c) - 0.5) / Y00] for c in cols])
    sc = hand_scene([(0, 0, z, 0.5) for z in zs], [np.log([s, s, s, 10.0])] * n, logit=logits, sh=sh, bg=bg)
    return sc, oracle_for(sc, cfg=cfg)


def _centre_alpha(sc, o, i):
    """alpha of splat i at pixel (31,31) (centre 31.5, 31.5) from its own 2D footprint."""
    p = o.prims()
    A, B, C = p.conic[i]
    dx, dy = p.uv[i, 0] - 31.5, p.uv[i, 1] - 31.5
    return p.opacity[i] * np.exp(-0.5 * (A * dx * dx + C * dy * dy) - B * dx * dy)


def test_two_layer_over_and_depth_swap():
    c1, c2 = (0.9, 0.1, 0.2), (0.2, 0.8, 0.6)
    sc, o = _layers([0.0, 1.0], [0.3, -0.4], [c1, c2], cfg=oracle.PURE_CFG, bg=(0.05, 0.05, 0.05))
    img = o.forward()[0]
    a1, a2 = _centre_alpha(sc, o, 0), _centre_alpha(sc, o, 1)
    ref = a1 * np.array(c1) + (1 - a1) * a2 * np.array(c2) + (1 - a1) * (1 - a2) * 0.05
    np.testing.assert_allclose(img[:, 31, 31], ref, atol=1e-14)
    # swapping the depths swaps who is in front ("sorted according to their depth", L83)
    sc2, o2 = _layers([1.0, 0.0], [0.3, -0.4], [c1, c2], cfg=oracle.PURE_CFG, bg=(0.05, 0.05, 0.05))
    b1, b2 = _centre_alpha(sc2, o2, 0), _centre_alpha(sc2, o2, 1)
    ref2 = b2 * np.array(c2) + (1 - b2) * b1 * np.array(c1) + (1 - b1) * (1 - b2) * 0.05
    np.testing.assert_allclose(o2.forward()[0][:, 31, 31], ref2, atol=1e-14)
    assert np.abs(ref - ref2).max() > 1e-2


def test_identical_layers_geometric_series():
    K = 6
    sc, o = _layers([0.0] * K, [-1.0] * K, [(0.7, 0.7, 0.7)] * K, cfg=oracle.PURE_CFG)
    img, fT, _, _ = o.forward()
    a = _centre_alpha(sc, o, 0)
    np.testing.assert_allclose(fT[31, 31], (1 - a) ** K, rtol=1e-13)
    np.testing.assert_allclose(img[:, 31, 31], 0.7 * (1 - (1 - a) ** K), rtol=1e-13)


def test_thresholds_alpha_clamp_skip_and_termination():
    # alpha clamp: an (almost) opaque splat is capped at 0.99
    sc, o = _layers([0.0], [20.0], [(1.0, 1.0, 1.0)], s=2.0)
    img, fT, nc, _ = o.forward()
    np.testing.assert_allclose(fT[31, 31], 0.01, rtol=1e-12)
    # termination: T after k splats of alpha .99 is .01^k; the third would give 1e-6 < 1e-4 and is NOT composited
    sc, o = _layers([0.0, 0.5, 1.0, 1.5], [20.0] * 4, [(1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 1)], s=2.0)
    img, fT, nc, _ = o.forward()
    np.testing.assert_allclose(img[:, 31, 31], [0.99, 0.01 * 0.99, 0.0], rtol=1e-12, atol=1e-15)
    assert nc[31, 31] == 2 and abs(fT[31, 31] - 1e-4) < 1e-15
    # skip: alpha < 1/255 contributes nothing and leaves T untouched
    sc, o = _layers([0.0], [np.log((1 / 300) / (1 - 1 / 300))], [(1, 1, 1)], s=2.0)
    img, fT, nc, _ = o.forward()
    assert img.max() == 0 and fT.min() == 1.0 and nc.max() == 0


def test_pure_eq6_direct_evaluation():
    """'pure eq. 6' mode against a direct numpy evaluation of eq. 6 over ALL primitives at every pixel."""
    sc = scenes.tiny()
    o = oracle_for(sc, cfg=oracle.PURE_CFG)
    p = o.prims()
    img = o.forward()[0]
    vis = np.where(p.status == oracle.STATUS_VISIBLE)[0]
    order = sorted(vis, key=lambda i: (int(np.float32(p.p_cam[i, 2]).view(np.uint32)), i))
    ys, xs = np.mgrid[0:64, 0:64] + 0.5
    T, out = np.ones((64, 64)), np.zeros((3, 64, 64))
    for i in order:
        dx, dy = p.uv[i, 0] - xs, p.uv[i, 1] - ys
        A, B, C = p.conic[i]
        a = p.opacity[i] * np.exp(np.minimum(0, -0.5 * (A * dx * dx + C * dy * dy) - B * dx * dy))
        out += p.rgb[i][:, None, None] * (a * T)[None]
        T *= 1 - a
    np.testing.assert_allclose(img, out, atol=1e-13)
    # truncated (default) renderer differs from pure eq. 6 only by the documented truncations (L147 "approximate")
    img_t = oracle_for(sc).forward()[0]
    assert 0 < np.abs(img_t - img).max() < 2e-2


# ------------------------------------------------------------------ whole-renderer invariants
def test_permutation_invariance():
    sc = scenes.tiny()
    img = oracle_for(sc).forward()[0]
    perm = np.random.default_rng(0).permutation(sc.N)
    img_p = oracle_for(sc.subset(perm)).forward()[0]
    np.testing.assert_allclose(img_p, img, atol=1e-15)        # no exact depth ties in this scene


def test_far_in_time_contributes_nothing():
    sc = scenes.tiny()
    img = oracle_for(sc).forward()[0]
    p = oracle_for(sc).prims()
    keep = np.where(p.status != oracle.STATUS_CULL_TIME)[0]
    assert 0 < len(keep) < sc.N
    img_k = oracle_for(sc.subset(keep)).forward()[0]
    assert np.array_equal(img_k, img)                          # bit-identical after removing time-culled primitives
    # |t - mu_t| >> sigma_t: invisible even with the filter off
    far = hand_scene([(0, 0, 0, 0.5)], [np.log([0.3, 0.3, 0.3, 0.01])], logit=[5.0], sh=[[[3, 3, 3]]], t=1.5)
    assert oracle_for(far, cfg=dict(marginal_min=0.0, alpha_min=0.0)).forward()[0].max() < 1e-300


def test_empty_and_all_culled():
    sc = hand_scene(np.zeros((0, 4)), np.zeros((0, 4)), quat_l=np.zeros((0, 4)), quat_r=np.zeros((0, 4)),
                    logit=np.zeros(0), sh=np.zeros((0, 1, 3)), bg=(0.2, 0.4, 0.6))
    img, fT, nc, _ = oracle_for(sc).forward()
    np.testing.assert_allclose(img, np.array([0.2, 0.4, 0.6])[:, None, None] * np.ones((3, 64, 64)))
    # behind the camera / non-finite / zero quaternion are culled, never poison the image
    sc = hand_scene([(0, 0, -10, 0.5), (0, 0, 0, 0.5), (0, 0, 0, 0.5)], [[-2] * 4, [np.nan, -2, -2, -2], [-2] * 4],
                    quat_l=[[1, 0, 0, 0], [1, 0, 0, 0], [0, 0, 0, 0]], quat_r=[[1, 0, 0, 0]] * 3)
    o = oracle_for(sc)
    assert list(o.prims().status) == [oracle.STATUS_CULL_NEAR, oracle.STATUS_CULL_NONFINITE, oracle.STATUS_CULL_NONFINITE]
    assert o.forward()[0].max() == 0


# ------------------------------------------------------------------ backward
PARAMS = ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")


def _loss_and_state(sc, G, cfg):
    o = oracle_for(sc, cfg=cfg)
    img, fT, nc, mg = o.forward()
    return float((img * G).sum()), o, nc, mg


def _fd_check(seed, cfg, tol=1e-5, N=8, sh_degree=1, n_time=2, scene=None, need_clamp=0):
    sc = scene if scene is not None else scenes.fd_scene(seed, N, sh_degree, n_time)
    for k in PARAMS:                       # promote to float64 so that +-h is representable
        setattr(sc, k, getattr(sc, k).astype(np.float64))
    G = scenes.upstream_normal(seed, 64, 64).astype(np.float64)
    L0, o0, nc0, mg0 = _loss_and_state(sc, G, cfg)
    p0 = o0.prims()
    assert (p0.status == 0).all()
    if need_clamp:                         # the guard-band clamped branch of J must be the one differentiated
        assert all((int(b) & need_clamp) for b in p0.clamp_bits), p0.clamp_bits
    if not cfg.get("full_support"):
        if mg0.min() < 1e-4 or p0.fragility.min() < 1e-4:
            return None                    # too close to a discontinuity: the caller resamples
    grads = o0.backward(G)
    lists0 = o0.tile_lists()
    worst = {}
    for name in PARAMS:
        arr = getattr(sc, name)
        fd = np.zeros_like(arr)
        it = np.nditer(arr, flags=["multi_index"])
        for x in it:
            idx = it.multi_index
            x0 = float(x)                      # x is a live view into arr: take the value before perturbing
            h = 1e-6 * max(1.0, abs(x0))
            vals = []
            for sgn in (+1, -1):
                arr[idx] = x0 + sgn * h
                Lp, op, ncp, _ = _loss_and_state(sc, G, cfg)
                # no discrete decision may change across +-h
                assert np.array_equal(ncp, nc0) and np.array_equal(op.tile_lists()[1], lists0[1])
                assert np.array_equal(op.prims().clamp_bits, p0.clamp_bits)
                vals.append(Lp)
            arr[idx] = x0
            fd[idx] = (vals[0] - vals[1]) / (2 * h)
        worst[name] = rel_l2(grads[name], fd)
        assert worst[name] < tol, (name, worst[name])
    return worst


# (L, n_time): the round-1 pin (1, 2); degree 2 alone; and the colour order every benchmark configuration runs, degree 3 x
# 3 Fourier orders (eq. 20, PAPER.md:L187 with Delta per L183) — the hand-derived gradient rows of Y_4..Y_15 and the n >= 2
# branch of the Delta-derivative are only reached here
@pytest.mark.parametrize("mode", ["default", "pure"])
@pytest.mark.parametrize("L,n_time,N", [(1, 2, 8), (2, 1, 6), (3, 3, 4)])
def test_backward_matches_central_differences(mode, L, n_time, N):
    cfg = dict(oracle.DEFAULT_CFG) if mode == "default" else dict(oracle.PURE_CFG)
    for seed in range(100, 120):
        res = _fd_check(seed, cfg, N=N, sh_degree=L, n_time=n_time)
        if res is not None:
            assert res["sh"] < 1e-5 and res["mean"] < 1e-5
            return
    pytest.fail("no finite-difference scene far from every threshold found")


def _clamp_scene(L=1, n_time=2):
    """Two large splats whose centres project OUTSIDE the guard band (|x/z| resp. |y/z| > 1.3 W / (2 fx) = 0.606 for the
    64x64, fov 50 camera at distance 4), so that J is evaluated at the clamped ratio
    while their 3-sigma support still reaches into the image: splat 0 clamps in x (bit 8), splat 1 in y (bit 16)."""
    K = n_time * (L + 1) ** 2
    rng = np.random.default_rng(7)
    sh = 0.05 * rng.standard_normal((2, K, 3))
    sh[:, 0, :] = 1.0 + 0.1 * rng.standard_normal((2, 3))
    ql = rng.standard_normal((2, 4)); qr = rng.standard_normal((2, 4))
    # a mild space-time tilt only: q_r = (a, b, c, -d) + noise keeps the splat near its spatial position at t
    qr = ql * np.array([1, 1, 1, -1]) + 0.1 * qr
    return hand_scene([(3.4, 0.2, 0.0, 0.45), (-0.3, -3.3, 0.3, 0.55)], [np.log([0.8, 0.7, 0.75, 0.6]), np.log([0.7, 0.8, 0.75, 0.6])],
                      quat_l=ql, quat_r=qr, logit=[0.4, -0.2], sh=sh, sh_degree=L, n_time=n_time, bg=(0.1, 0.2, 0.3))


@pytest.mark.parametrize("mode", ["default", "pure"])
def test_backward_with_the_guard_band_clamp_active(mode):
    """The clamped-J branch of the forward and of backward_one ('x' = lim z => that entry is
    -fx lim / z') against central differences; _fd_check asserts that the clamp bits are set and identical at +-h."""
    cfg = dict(oracle.DEFAULT_CFG) if mode == "default" else dict(oracle.PURE_CFG)
    sc = _clamp_scene()
    o = oracle_for(sc, cfg=cfg)
    bits = o.prims().clamp_bits.astype(int)
    assert bits[0] & 8 and bits[1] & 16, bits
    img = o.forward()[0]
    assert img.max() > 0.3 and (np.abs(img - np.array([0.1, 0.2, 0.3])[:, None, None]).max(0) > 1e-3).mean() > 0.2   # the splats are on screen
    res = _fd_check(0, cfg, scene=sc, need_clamp=24)
    assert res is not None and max(res.values()) < 1e-5, res
    # and the clamp matters: the unclamped Jacobian gives a different footprint (guard = 100 disables the clamp)
    o2 = oracle_for(sc, cfg=dict(cfg, guard=100.0))
    assert not (o2.prims().clamp_bits.astype(int) & 24).any()
    assert np.abs(o2.prims().conic - o.prims().conic).max() > 1e-4


def test_backward_invariants():
    sc = scenes.tiny()
    G = scenes.upstream_normal(0, 64, 64)
    o = oracle_for(sc)
    o.forward()
    g = o.backward(G)
    p = o.prims()
    culled = p.status != 0
    for k in PARAMS:
        assert np.abs(g[k][culled]).max() == 0                 # dL/dparams = 0 for culled primitives
        assert np.abs(g[k][~culled]).max() > 0
    # scale invariance of the normalised quaternions: q . dL/dq = 0
    for k in ("quat_l", "quat_r"):
        q = getattr(sc, k).astype(np.float64)
        dots = np.abs((q * g[k]).sum(1))
        assert dots.max() < 1e-12 * max(1.0, np.abs(g[k]).max())
    # accumulation semantics: a second backward call adds onto the same arrays
    g2 = o.backward(2.0 * G)
    np.testing.assert_allclose(g2["mean"], 2 * g["mean"], rtol=1e-12, atol=1e-300)


def test_backward_through_active_clamps_is_zero():
    # alpha at alpha_max: zero slope wrt opacity and geometry, colour gradient still flows (reading S16)
    sc, G = None, np.ones((3, 64, 64))
    sc = hand_scene([(0, 0, 0, 0.5)], [np.log([50.0, 50.0, 50.0, 10.0])], logit=[20.0], sh=[[[1.0, 1.0, 1.0]]])
    o = oracle_for(sc)
    o.forward()
    g = o.backward(G)
    assert g["g9"][0, 5] == 0 and np.abs(g["g9"][0, :5]).max() == 0 and g["g9"][0, 6] > 0
    # colour clamped at 0: no gradient to the coefficients of that channel
    sc = hand_scene([(0, 0, 0, 0.5)], [np.log([0.3, 0.3, 0.3, 10.0])], sh=[[[-5.0, 1.0, 1.0]]])
    o = oracle_for(sc)
    o.forward()
    g = o.backward(G)
    assert g["sh"][0, 0, 0] == 0 and g["sh"][0, 0, 1] != 0
