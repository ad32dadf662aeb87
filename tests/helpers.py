"""Shared test helpers: build an oracle from a Scene, small hand-made scenes."""
import numpy as np

import oracle
from paper_2412_20720_b200 import scenes


def make_oracle(scene):
    return oracle.Oracle(**scene.arrays(), sh_degree=scene.sh_degree, n_time=scene.n_time)


def run_pre(o, view, cfg=None, t=None):
    o.preprocess(view.view, (view.fx, view.fy, view.cx, view.cy), view.width, view.height,
                 view.t if t is None else t, view.period_T, view.bg, cfg)
    return o


def oracle_for(scene, view_index=0, cfg=None, t=None):
    o = make_oracle(scene)
    return run_pre(o, scene.views[view_index], cfg, t)


def hand_scene(mean, log_scale, quat_l=None, quat_r=None, logit=None, sh=None, sh_degree=0, n_time=1,
               width=64, height=64, fov=50.0, cam_z=4.0, t=0.5, T=1.0, bg=(0, 0, 0)):
    """A scene from explicit arrays with a camera at (0,0,-cam_z) looking +z."""
    mean = np.atleast_2d(np.asarray(mean, dtype=np.float64))
    N = mean.shape[0]
    K = n_time * (sh_degree + 1) ** 2
    ident = np.tile(np.array([1.0, 0, 0, 0]), (N, 1))
    quat_l = ident if quat_l is None else np.atleast_2d(quat_l)
    quat_r = ident if quat_r is None else np.atleast_2d(quat_r)
    logit = np.zeros(N) if logit is None else np.atleast_1d(logit)
    sh = np.zeros((N, K, 3)) if sh is None else np.asarray(sh, dtype=np.float64).reshape(N, K, 3)
    fx = 0.5 * width / np.tan(np.deg2rad(0.5 * fov))
    V = np.eye(4)
    V[2, 3] = cam_z
    view = scenes.View(V, fx, fx, 0.5 * width, 0.5 * height, width, height, t, T, bg)
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    return scenes.Scene("hand", sh_degree, n_time, f(mean), f(np.atleast_2d(log_scale)), f(quat_l), f(quat_r),
                        f(logit), f(sh), [view], 0)


def rel_l2(a, b):
    a, b = np.asarray(a, dtype=np.float64).ravel(), np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))
