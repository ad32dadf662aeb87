"""Seeded synthetic scenes and cameras shaped like the paper's workloads (BASELINE.json configs 1-5).

This module holds NO arithmetic of the method: it only draws parameter arrays, camera matrices,
query times and upstream gradients / target images.  It is the one module both the CUDA-path tests
and the oracle-path tests use.  Every attribute of primitive ``i`` is a pure function of
(seed, stream, i): a SplitMix64-style counter hash -> uniform -> Box-Muller, so any subset of a
scene can be regenerated independently and N can grow without changing earlier primitives.

Stand-ins: cfg2 <-> D-NeRF, cfg3/cfg5 <-> Plenoptic
Video (L324-L326, Table 7), cfg4 <-> Waymo-NOTR clips (L572-L587).  None of those datasets is read.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = x + np.uint64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return x ^ (x >> np.uint64(31))


def uniform(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """U[0,1) float64, element i a pure function of (seed, stream, start+i)."""
    idx = np.arange(start, start + n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _mix(np.uint64(seed) * np.uint64(0xD1342543DE82EF95) + np.uint64(stream) * np.uint64(0xA0761D6478BD642F) + np.uint64(1))
        h = _mix(_mix(idx ^ key) + key)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """N(0,1) float64 by Box-Muller on two counter streams."""
    u1 = uniform(seed, 2 * stream + 1000003, n, start)
    u2 = uniform(seed, 2 * stream + 1000004, n, start)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


@dataclass
class View:
    view: np.ndarray          # [4,4] float32 world->camera, +z forward
    fx: float
    fy: float
    cx: float
    cy: float
    width: int
    height: int
    t: float
    period_T: float
    bg: tuple = (0.0, 0.0, 0.0)

    def as_fp32(self) -> "View":
        """The boundary takes fp32 scalars: a copy whose scalars are fp32-representable, so that the CUDA path and the
        float64 oracle receive bit-identical inputs.  All generators below return such views."""
        r = lambda x: float(np.float32(x))
        return View(np.asarray(self.view, dtype=np.float32), r(self.fx), r(self.fy), r(self.cx), r(self.cy), self.width, self.height,
                    r(self.t), r(self.period_T), tuple(r(b) for b in self.bg))


@dataclass
class Scene:
    name: str
    sh_degree: int
    n_time: int
    mean: np.ndarray          # [N,4] float32 (x,y,z,t)
    log_scale: np.ndarray     # [N,4]
    quat_l: np.ndarray        # [N,4]
    quat_r: np.ndarray        # [N,4]
    opacity_logit: np.ndarray # [N]
    sh: np.ndarray            # [N,K,3]
    views: List[View] = field(default_factory=list)
    seed: int = 0

    @property
    def N(self) -> int:
        return int(self.mean.shape[0])

    @property
    def K(self) -> int:
        return self.n_time * (self.sh_degree + 1) ** 2

    def arrays(self):
        return dict(mean=self.mean, log_scale=self.log_scale, quat_l=self.quat_l, quat_r=self.quat_r,
                    opacity_logit=self.opacity_logit, sh=self.sh)

    def subset(self, idx) -> "Scene":
        return Scene(self.name, self.sh_degree, self.n_time, self.mean[idx].copy(), self.log_scale[idx].copy(),
                     self.quat_l[idx].copy(), self.quat_r[idx].copy(), self.opacity_logit[idx].copy(),
                     self.sh[idx].copy(), list(self.views), self.seed)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _normalise(q):
    return q / np.linalg.norm(q, axis=1, keepdims=True)


def _quats(seed, N, mode):
    ql = _normalise(np.stack([normal(seed, 20 + k, N) for k in range(4)], axis=1))
    if mode == "random":        # cfg1: fully random 4D rotations (both quaternions = normalised N(0,I4))
        qr = _normalise(np.stack([normal(seed, 24 + k, N) for k in range(4)], axis=1))
    elif mode == "tilted":      # cfg2-5: random spatial orientation with a small space-time tilt
        base = ql * np.array([1.0, 1.0, 1.0, -1.0])
        qr = _normalise(base + 0.1 * np.stack([normal(seed, 24 + k, N) for k in range(4)], axis=1))
    else:
        raise ValueError(mode)
    return ql, qr


def _sh_coeffs(seed, N, K):
    """DC (k=0) ~ N(0.5, 0.2), all other coefficients ~ N(0, 0.05) (BASELINE.json cfg1, reused for cfg2-5)."""
    sh = 0.05 * normal(seed, 40, N * K * 3).reshape(N, K, 3)
    sh[:, 0, :] = 0.5 + 0.2 * normal(seed, 41, N * 3).reshape(N, 3)
    return sh


def _pinhole(width, height, fov_x_deg):
    fx = 0.5 * width / np.tan(np.deg2rad(0.5 * fov_x_deg))
    return float(fx), float(fx), 0.5 * width, 0.5 * height


def _look_at(cam_pos, target):
    """world->camera with +z forward, +x right, +y down."""
    f = target - cam_pos
    f = f / np.linalg.norm(f)
    up = np.array([0.0, -1.0, 0.0])
    r = np.cross(up, f)
    if np.linalg.norm(r) < 1e-6:
        r = np.array([1.0, 0.0, 0.0])
    r = r / np.linalg.norm(r)
    d = np.cross(f, r)
    Wm = np.stack([r, d, f], axis=0)
    V = np.eye(4)
    V[:3, :3] = Wm
    V[:3, 3] = -Wm @ cam_pos
    return V


def _axis_angle(axis, ang):
    axis = axis / np.linalg.norm(axis)
    Kx = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
    return np.eye(3) + np.sin(ang) * Kx + (1 - np.cos(ang)) * (Kx @ Kx)


def tiny(seed: int = 0, N: int = 256) -> Scene:
    """cfg1: N=256, 64x64, fov 50 deg, camera 4 units from the origin, t=0.5, L=1, n_time=2."""
    mean = np.stack([2 * uniform(seed, 1, N) - 1, 2 * uniform(seed, 2, N) - 1, 2 * uniform(seed, 3, N) - 1,
                     uniform(seed, 4, N)], axis=1)
    ls = np.stack([-3 + 0.3 * normal(seed, 10 + k, N) for k in range(3)] + [-1.5 + 0.3 * normal(seed, 13, N)], axis=1)
    ql, qr = _quats(seed, N, "random")
    logit = normal(seed, 30, N)
    sh = _sh_coeffs(seed, N, 8)
    fx, fy, cx, cy = _pinhole(64, 64, 50.0)
    V = np.eye(4)
    V[2, 3] = 4.0      # camera at (0,0,-4) looking +z at the origin
    view = View(_f32(V), fx, fy, cx, cy, 64, 64, 0.5, 1.0).as_fp32()
    return Scene("cfg1_tiny", 1, 2, _f32(mean), _f32(ls), _f32(ql), _f32(qr), _f32(logit), _f32(sh), [view], seed)


def single_object(seed: int = 2, N: int = 100_000, width: int = 800, height: int = 800) -> Scene:
    """cfg2: N=100k in the unit ball x t in [0,1], L=3, n_time=3, 800x800 fov 40, camera on a sphere r=4."""
    d = np.stack([normal(seed, 1 + k, N) for k in range(3)], axis=1)
    d = d / np.linalg.norm(d, axis=1, keepdims=True)
    rad = uniform(seed, 5, N) ** (1.0 / 3.0)
    mean = np.concatenate([d * rad[:, None], uniform(seed, 4, N)[:, None]], axis=1)
    ls = np.stack([-4.5 + 0.5 * normal(seed, 10 + k, N) for k in range(3)] + [-2 + 0.5 * normal(seed, 13, N)], axis=1)
    ql, qr = _quats(seed, N, "tilted")
    logit = normal(seed, 30, N)
    sh = _sh_coeffs(seed, N, 48)
    fx, fy, cx, cy = _pinhole(width, height, 40.0)
    az = 2 * np.pi * uniform(seed, 50, 1)[0]
    el = np.deg2rad(-30 + 60 * uniform(seed, 51, 1)[0])
    cam = 4.0 * np.array([np.cos(el) * np.sin(az), np.sin(el), -np.cos(el) * np.cos(az)])
    t = float(uniform(seed, 52, 1)[0])
    view = View(_f32(_look_at(cam, np.zeros(3))), fx, fy, cx, cy, width, height, t, 1.0).as_fp32()
    return Scene("cfg2_object", 3, 3, _f32(mean), _f32(ls), _f32(ql), _f32(qr), _f32(logit), _f32(sh), [view], seed)


def _video_params(seed, N, quat_mode="tilted"):
    mean = np.stack([-3 + 6 * uniform(seed, 1, N), -2 + 4 * uniform(seed, 2, N), 2 + 6 * uniform(seed, 3, N),
                     10 * uniform(seed, 4, N)], axis=1)
    ls = np.stack([-4 + 0.6 * normal(seed, 10 + k, N) for k in range(3)] + [-0.5 + 0.7 * normal(seed, 13, N)], axis=1)
    ql, qr = _quats(seed, N, quat_mode)
    logit = normal(seed, 30, N)
    sh = _sh_coeffs(seed, N, 48)
    return mean, ls, ql, qr, logit, sh


def multiview_video(seed: int = 3, N: int = 1_000_000, width: int = 1352, height: int = 1014, n_views: int = 4,
                    quat_mode: str = "tilted") -> Scene:
    """cfg3: N=1M in [-3,3]x[-2,2]x[2,8] (camera frame) x t in [0,10], T=10, 1352x1014 fov 60, 4 jittered views."""
    mean, ls, ql, qr, logit, sh = _video_params(seed, N, quat_mode)
    fx, fy, cx, cy = _pinhole(width, height, 60.0)
    views = []
    for k in range(n_views):
        trans = 0.1 * normal(seed, 60 + k, 3)
        axis = normal(seed, 70 + k, 3)
        ang = np.deg2rad(2.0) * normal(seed, 80 + k, 1)[0]
        V = np.eye(4)
        V[:3, :3] = _axis_angle(axis, ang)
        V[:3, 3] = trans
        t = 10.0 * float(uniform(seed, 90 + k, 1)[0])
        views.append(View(_f32(V), fx, fy, cx, cy, width, height, t, 10.0).as_fp32())
    return Scene("cfg3_video", 3, 3, _f32(mean), _f32(ls), _f32(ql), _f32(qr), _f32(logit), _f32(sh), views, seed)


def driving(seed: int = 4, N: int = 3_000_000, width: int = 1920, height: int = 1280, n_views: int = 3) -> Scene:
    """cfg4: N=3M in a 20x10x100 m corridor x t in [0,20], 70% long-lived / 30% transient, L=3, n_time=2."""
    mean = np.stack([-10 + 20 * uniform(seed, 1, N), -5 + 10 * uniform(seed, 2, N), 100 * uniform(seed, 3, N),
                     20 * uniform(seed, 4, N)], axis=1)
    long_lived = uniform(seed, 14, N) < 0.7
    ls_t = np.where(long_lived, 2 + 0.3 * normal(seed, 13, N), -1 + 0.5 * normal(seed, 15, N))
    ls = np.stack([-2.5 + 0.8 * normal(seed, 10 + k, N) for k in range(3)] + [ls_t], axis=1)
    ql, qr = _quats(seed, N, "tilted")
    logit = normal(seed, 30, N)
    sh = _sh_coeffs(seed, N, 32)
    fx, fy, cx, cy = _pinhole(width, height, 60.0)
    views = []
    for k in range(n_views):
        t = 20.0 * float(uniform(seed, 90 + k, 1)[0])
        V = np.eye(4)
        V[2, 3] = -(10.0 + 4.0 * t)     # camera at (0,0,10+4t) looking +z
        views.append(View(_f32(V), fx, fy, cx, cy, width, height, t, 20.0).as_fp32())
    return Scene("cfg4_driving", 3, 2, _f32(mean), _f32(ls), _f32(ql), _f32(qr), _f32(logit), _f32(sh), views, seed)


def sweep(seed: int = 3, N: int = 1_000_000, width: int = 1352, height: int = 1014, n_frames: int = 120) -> Scene:
    """cfg5: cfg3 distributions, fixed base camera, n_frames query times evenly spaced over [0,10]."""
    mean, ls, ql, qr, logit, sh = _video_params(seed, N)
    fx, fy, cx, cy = _pinhole(width, height, 60.0)
    views = [View(_f32(np.eye(4)), fx, fy, cx, cy, width, height, 10.0 * k / max(1, n_frames - 1), 10.0).as_fp32()
             for k in range(n_frames)]
    return Scene("cfg5_sweep", 3, 3, _f32(mean), _f32(ls), _f32(ql), _f32(qr), _f32(logit), _f32(sh), views, seed)


def upstream_normal(seed: int, width: int, height: int) -> np.ndarray:
    """cfg1's upstream dL/dimage ~ N(0,1), [3,H,W] float32."""
    return _f32(normal(seed, 200, 3 * width * height).reshape(3, height, width))


def target_image(seed: int, view_index: int, width: int, height: int) -> np.ndarray:
    """Seeded random target image ~ U[0,1), [3,H,W] float32 (cfg2-4's L1 loss target)."""
    return _f32(uniform(seed, 300 + view_index, 3 * width * height).reshape(3, height, width))


def fd_scene(seed: int, N: int = 8, sh_degree: int = 1, n_time: int = 2) -> Scene:
    """Finite-difference scenes: <=8 large, translucent splats far from every threshold; K = n_time (L+1)^2
    colour coefficients per channel (the defaults give the K = 8 scenes of round 1 unchanged)."""
    K = n_time * (sh_degree + 1) ** 2
    mean = np.stack([uniform(seed, 1, N) - 0.5, uniform(seed, 2, N) - 0.5, uniform(seed, 3, N) - 0.5,
                     0.5 + 0.3 * (uniform(seed, 4, N) - 0.5)], axis=1)
    ls = np.stack([-1.5 + 0.2 * normal(seed, 10 + k, N) for k in range(3)] + [-0.5 + 0.2 * normal(seed, 13, N)], axis=1)
    ql, qr = _quats(seed, N, "random")
    ql = ql * (0.5 + uniform(seed, 28, N))[:, None]     # non-unit on purpose: normalisation is inside
    qr = qr * (0.5 + uniform(seed, 29, N))[:, None]
    logit = 0.5 * normal(seed, 30, N)
    sh = 0.05 * normal(seed, 40, N * K * 3).reshape(N, K, 3)
    sh[:, 0, :] = 1.0 + 0.1 * normal(seed, 41, N * 3).reshape(N, 3)
    fx, fy, cx, cy = _pinhole(64, 64, 50.0)
    V = np.eye(4)
    V[:3, :3] = _axis_angle(np.array([0.3, 1.0, 0.2]), 0.2)
    V[:3, 3] = np.array([0.1, -0.05, 4.0])
    view = View(_f32(V), fx, fy, cx, cy, 64, 64, 0.5, 1.0, (0.1, 0.2, 0.3)).as_fp32()
    return Scene("fd", sh_degree, n_time, _f32(mean), _f32(ls), _f32(ql), _f32(qr), _f32(logit), _f32(sh), [view], seed)


def compact_model(seed: int = 6, N: int = 1_000_000, sh_degree: int = 3, n_time: int = 3, rvq=((6, 64), (6, 64), (6, 64), (8, 256))) -> dict:
    """Seeded stand-in for a compact model: codebook sizes of section 8.3.1 (scale 6x64, both
    quaternions share 6x64, base colour 6x64, rest 8x256), uniformly random indices, binary16 positions in cfg3's box,
    8-bit opacity codes over the logit range [-4, 6].  Stage s of a codebook holds values ~ N(centre_s, (spread / 2^s)):
    the first stage carries the parameter's scale, later stages shrinking residuals, as a fitted residual VQ would.
    Holds no arithmetic of the method — only random tables and indices."""
    K = n_time * (sh_degree + 1) ** 2
    (s_st, s_en), (r_st, r_en), (d_st, d_en), (c_st, c_en) = rvq

    def book(stream, stages, entries, dim, centre, spread):
        cb = normal(seed, stream, stages * entries * dim).reshape(stages, entries, dim) * spread
        cb = cb / (2.0 ** np.arange(stages))[:, None, None]
        cb[0] += np.asarray(centre, dtype=np.float64)
        return _f32(cb)

    def indices(stream, stages, entries):
        return np.ascontiguousarray(np.minimum((uniform(seed, stream, N * stages) * entries).astype(np.int64), entries - 1)
                                    .reshape(N, stages).astype(np.uint8))

    mean = np.stack([-3 + 6 * uniform(seed, 1, N), -2 + 4 * uniform(seed, 2, N), 2 + 6 * uniform(seed, 3, N),
                     10 * uniform(seed, 4, N)], axis=1)
    out = dict(mean_f16=np.ascontiguousarray(mean.astype(np.float16)),
               opacity_code=np.minimum((uniform(seed, 5, N) * 256).astype(np.int64), 255).astype(np.uint8),
               opacity_lo=-4.0, opacity_hi=6.0, opacity_bits=8,
               scale_cb=book(100, s_st, s_en, 4, [-4.0, -4.0, -4.0, -0.5], 0.6), scale_idx=indices(101, s_st, s_en),
               rot_cb=book(110, r_st, r_en, 4, [0.0, 0.0, 0.0, 0.0], 1.0), rot_l_idx=indices(111, r_st, r_en),
               rot_r_idx=indices(112, r_st, r_en),
               dc_cb=book(120, d_st, d_en, 3, [0.5, 0.5, 0.5], 0.2), dc_idx=indices(121, d_st, d_en),
               rest_cb=None, rest_idx=None)
    if K > 1:
        out["rest_cb"] = book(130, c_st, c_en, (K - 1) * 3, np.zeros((K - 1) * 3), 0.05)
        out["rest_idx"] = indices(131, c_st, c_en)
    return out
