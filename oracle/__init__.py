"""float64 CPU ORACLE for the 4D-Gaussian time-sliced tile rasterizer (arxiv 2412.20720).

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` leg may import this package.  It shares no code with the
CUDA path under ``paper_2412_20720_b200/`` and never imports it.

The arithmetic lives in ``fdgs_oracle.cpp`` (plain C++17, float64, step by step in the paper's
order); this module only builds it with g++ and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fdgs_oracle.cpp")
_LIB = os.path.join(_HERE, "libfdgs_oracle.so")
_lib = None

STATUS_VISIBLE, STATUS_CULL_TIME, STATUS_CULL_NEAR, STATUS_CULL_RECT, STATUS_CULL_NONFINITE = range(5)

# default thresholds (readings S7/S8): marginal_min, alpha_min, alpha_max,
# transmittance_min, dilation, cutoff_sigma, znear, guard
DEFAULT_CFG = dict(marginal_min=0.05, alpha_min=1.0 / 255.0, alpha_max=0.99, transmittance_min=1e-4,
                   dilation=0.3, cutoff_sigma=3.0, znear=0.2, guard=1.3, full_support=0)
# "pure eq. 6" mode: no truncation at all, every primitive evaluated at every pixel
PURE_CFG = dict(marginal_min=0.0, alpha_min=0.0, alpha_max=1.0, transmittance_min=0.0,
                dilation=0.3, cutoff_sigma=3.0, znear=0.2, guard=1.3, full_support=1)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2 -fopenmp).  Returns the path of the shared library.
    FDGS_ORACLE_SANITIZE=1 builds and loads an -fsanitize=address,undefined variant instead; run the
    CPU suite under it with
        FDGS_ORACLE_SANITIZE=1 LD_PRELOAD=$(g++ -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
            python -m pytest tests -m "not gpu" -q"""
    lib, extra = _LIB, []
    if os.environ.get("FDGS_ORACLE_SANITIZE"):
        lib = os.path.join(_HERE, "libfdgs_oracle_san.so")
        extra = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++17", "-ffp-contract=off", *extra, _SRC, "-o", lib]
        subprocess.run(cmd, check=True)
    return lib


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    lib.fdgs_oracle_create.restype = C.c_void_p
    lib.fdgs_oracle_create.argtypes = [C.c_int, C.c_int, C.c_int, dp, dp, dp, dp, dp, dp]
    lib.fdgs_oracle_destroy.argtypes = [C.c_void_p]
    lib.fdgs_oracle_preprocess.restype = C.c_int
    lib.fdgs_oracle_preprocess.argtypes = [C.c_void_p, dp, dp, C.c_int, C.c_int, C.c_double, C.c_double, dp, dp]
    lib.fdgs_oracle_num_pairs.restype = C.c_int64
    lib.fdgs_oracle_num_pairs.argtypes = [C.c_void_p]
    lib.fdgs_oracle_num_tiles.restype = C.c_int
    lib.fdgs_oracle_num_tiles.argtypes = [C.c_void_p]
    lib.fdgs_oracle_get_tile_lists.argtypes = [C.c_void_p, lp, ip]
    lib.fdgs_oracle_get_prims.argtypes = [C.c_void_p, dp]
    lib.fdgs_oracle_get_rot_cov.argtypes = [C.c_void_p, C.c_int, dp, dp]
    lib.fdgs_oracle_sh_basis.argtypes = [C.c_int, dp, dp]
    lib.fdgs_oracle_sh_basis_grad.argtypes = [C.c_int, dp, dp, dp]
    lib.fdgs_oracle_forward.argtypes = [C.c_void_p, dp, dp, ip, dp]
    lib.fdgs_oracle_backward.argtypes = [C.c_void_p, dp] + [dp] * 8
    lib.fdgs_oracle_get_depth_map.argtypes = [C.c_void_p, dp]
    lib.fdgs_oracle_backward_aux.argtypes = [C.c_void_p, dp, dp, dp] + [dp] * 10
    lib.fdgs_oracle_set_colour_override.argtypes = [C.c_void_p, dp]
    lib.fdgs_oracle_num_threads.restype = C.c_int
    lib.fdgs_oracle_set_num_threads.argtypes = [C.c_int]
    _lib = lib
    return lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def num_threads() -> int:
    return int(_load().fdgs_oracle_num_threads())


def set_num_threads(n: int) -> None:
    """OpenMP threads of the following calls (bench.py's single-thread / all-core CPU baseline)."""
    _load().fdgs_oracle_set_num_threads(int(n))


def sh_basis(sh_degree: int, direction) -> np.ndarray:
    d = np.ascontiguousarray(direction, dtype=np.float64)
    Y = np.zeros((sh_degree + 1) ** 2, dtype=np.float64)
    _load().fdgs_oracle_sh_basis(int(sh_degree), _d(d), _d(Y))
    return Y


def sh_basis_grad(sh_degree: int, direction):
    """(Y[(L+1)^2], dY/d(x,y,z)[(L+1)^2,3]) of the polynomial extension, as the oracle's backward uses them."""
    d = np.ascontiguousarray(direction, dtype=np.float64)
    K = (sh_degree + 1) ** 2
    Y, G = np.zeros(K, dtype=np.float64), np.zeros((K, 3), dtype=np.float64)
    _load().fdgs_oracle_sh_basis_grad(int(sh_degree), _d(d), _d(Y), _d(G))
    return Y, G


@dataclass
class Prims:
    """Per-primitive products of the oracle's preprocess (NaN where an earlier cull stopped the chain)."""
    raw: np.ndarray
    status: np.ndarray = field(init=False)

    def __post_init__(self):
        self.status = self.raw[:, 0].astype(np.int32)

    w = property(lambda s: s.raw[:, 1])
    sigma44 = property(lambda s: s.raw[:, 2])
    delta = property(lambda s: s.raw[:, 3])
    mu_c = property(lambda s: s.raw[:, 4:7])
    sigma_c6 = property(lambda s: s.raw[:, 7:13])
    p_cam = property(lambda s: s.raw[:, 13:16])
    uv = property(lambda s: s.raw[:, 16:18])
    conic = property(lambda s: s.raw[:, 18:21])
    radius = property(lambda s: s.raw[:, 21])
    rect = property(lambda s: s.raw[:, 22:26])
    rgb = property(lambda s: s.raw[:, 26:29])
    clamp_bits = property(lambda s: s.raw[:, 29])
    opacity = property(lambda s: s.raw[:, 30])
    depth32 = property(lambda s: s.raw[:, 31])
    fragility = property(lambda s: s.raw[:, 32])
    raw_rgb = property(lambda s: s.raw[:, 33:36])
    sigma2d = property(lambda s: s.raw[:, 36:39])

    def sigma_c(self, i) -> np.ndarray:
        xx, xy, xz, yy, yz, zz = self.raw[i, 7:13]
        return np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]])


class Oracle:
    """One scene (the six parameter arrays) loaded into the float64 oracle."""

    def __init__(self, mean, log_scale, quat_l, quat_r, opacity_logit, sh, sh_degree: int, n_time: int):
        lib = _load()
        f = lambda a: np.ascontiguousarray(np.asarray(a, dtype=np.float64))
        self.mean, self.log_scale, self.quat_l, self.quat_r = f(mean), f(log_scale), f(quat_l), f(quat_r)
        self.opacity_logit, self.sh = f(opacity_logit), f(sh)
        self.N = int(self.mean.shape[0])
        self.sh_degree, self.n_time = int(sh_degree), int(n_time)
        self.K = self.n_time * (self.sh_degree + 1) ** 2
        assert self.mean.shape == (self.N, 4) and self.log_scale.shape == (self.N, 4)
        assert self.quat_l.shape == (self.N, 4) and self.quat_r.shape == (self.N, 4)
        assert self.opacity_logit.shape == (self.N,) and self.sh.shape == (self.N, self.K, 3)
        self._h = lib.fdgs_oracle_create(self.N, self.sh_degree, self.n_time, _d(self.mean), _d(self.log_scale),
                                         _d(self.quat_l), _d(self.quat_r), _d(self.opacity_logit), _d(self.sh))
        if not self._h:
            raise ValueError("fdgs_oracle_create rejected the arguments")
        self.width = self.height = 0

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.fdgs_oracle_destroy(self._h)
            self._h = None

    def preprocess(self, view, intr, width, height, t, period_T, bg=(0, 0, 0), cfg=None):
        """view: 4x4 world->camera; intr: (fx,fy,cx,cy).  Runs the per-primitive chain and builds tile lists."""
        c = dict(DEFAULT_CFG)
        c.update(cfg or {})
        cfg9 = np.array([c["marginal_min"], c["alpha_min"], c["alpha_max"], c["transmittance_min"], c["dilation"],
                         c["cutoff_sigma"], c["znear"], c["guard"], float(c["full_support"])], dtype=np.float64)
        v = np.ascontiguousarray(np.asarray(view, dtype=np.float64).reshape(16))
        k = np.ascontiguousarray(np.asarray(intr, dtype=np.float64).reshape(4))
        b = np.ascontiguousarray(np.asarray(bg, dtype=np.float64).reshape(3))
        rc = _load().fdgs_oracle_preprocess(self._h, _d(v), _d(k), int(width), int(height), float(t), float(period_T),
                                            _d(b), _d(cfg9))
        if rc != 0:
            raise ValueError("fdgs_oracle_preprocess failed")
        self.width, self.height = int(width), int(height)
        return self

    def prims(self) -> Prims:
        out = np.zeros((self.N, 40), dtype=np.float64)
        _load().fdgs_oracle_get_prims(self._h, _d(out))
        return Prims(out)

    def rot_cov(self, i):
        R, S = np.zeros((4, 4)), np.zeros((4, 4))
        _load().fdgs_oracle_get_rot_cov(self._h, int(i), _d(R), _d(S))
        return R, S

    def tile_lists(self):
        """(tile_off[tiles+1] int64, tile_ids[D] int32): per tile, ids sorted by (fp32 depth bits, id)."""
        lib = _load()
        tiles, D = lib.fdgs_oracle_num_tiles(self._h), lib.fdgs_oracle_num_pairs(self._h)
        off, ids = np.zeros(tiles + 1, dtype=np.int64), np.zeros(max(D, 1), dtype=np.int32)
        lib.fdgs_oracle_get_tile_lists(self._h, off.ctypes.data_as(C.POINTER(C.c_int64)),
                                       ids.ctypes.data_as(C.POINTER(C.c_int32)))
        return off, ids[:D]

    def forward(self):
        """Returns image[3,H,W], final_T[H,W], n_contrib[H,W] (int32), margin[H,W]."""
        H, W = self.height, self.width
        img, fT = np.zeros((3, H, W)), np.zeros((H, W))
        nc, mg = np.zeros((H, W), dtype=np.int32), np.zeros((H, W))
        _load().fdgs_oracle_forward(self._h, _d(img), _d(fT), nc.ctypes.data_as(C.POINTER(C.c_int32)), _d(mg))
        return img, fT, nc, mg

    def depth_map(self):
        """Requires forward().  Auxiliary channel: rendered depth sum_k z_k alpha_k T_k, [H,W]."""
        out = np.zeros((self.height, self.width))
        _load().fdgs_oracle_get_depth_map(self._h, _d(out))
        return out

    def backward(self, dL_dimage, dL_ddepth=None, dL_dopacity=None, densify=None):
        """Requires forward().  Returns a dict of gradient arrays (float64) incl. 'mean2d', 'g9' and 'gz'.
        dL_ddepth / dL_dopacity [H,W]: upstream gradients of the auxiliary depth map and of O = 1 - final_T.
        densify: float64 [N,3] accumulated into (+=): |dL/d(u,v)|, |dL/dmu_t|, visibility count."""
        g = np.ascontiguousarray(np.asarray(dL_dimage, dtype=np.float64))
        assert g.shape == (3, self.height, self.width)
        aux = []
        for a in (dL_ddepth, dL_dopacity):
            if a is not None:
                a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
                assert a.shape == (self.height, self.width)
            aux.append(a)
        out = dict(mean=np.zeros((self.N, 4)), log_scale=np.zeros((self.N, 4)), quat_l=np.zeros((self.N, 4)),
                   quat_r=np.zeros((self.N, 4)), opacity_logit=np.zeros(self.N), sh=np.zeros((self.N, self.K, 3)),
                   mean2d=np.zeros((self.N, 2)), g9=np.zeros((self.N, 9)), gz=np.zeros(self.N))
        null = C.POINTER(C.c_double)()
        _load().fdgs_oracle_backward_aux(self._h, _d(g), _d(aux[0]) if aux[0] is not None else null,
                                         _d(aux[1]) if aux[1] is not None else null, _d(out["mean"]), _d(out["log_scale"]),
                                         _d(out["quat_l"]), _d(out["quat_r"]), _d(out["opacity_logit"]), _d(out["sh"]),
                                         _d(out["mean2d"]), _d(out["g9"]), _d(out["gz"]),
                                         _d(densify) if densify is not None else null)
        return out

    # ---- feature channels and rendered optical flow (L410) ------------------------------------------
    def _override(self, feat, c0):
        """Channels c0..c0+2 of feat[N,C] become the composited 'colour' of the visible primitives (zero padded)."""
        F = np.zeros((self.N, 3))
        n = min(3, feat.shape[1] - c0)
        F[:, :n] = feat[:, c0:c0 + n]
        _load().fdgs_oracle_set_colour_override(self._h, _d(np.ascontiguousarray(F)))
        return n

    def render_features(self, feat):
        """feat[N,C] -> F[C,H,W] = sum_k f_k alpha_k T_k: eq. 6 with the colour replaced by the feature vector, three
        channels per pass over the same tile lists.  Call preprocess() with bg = 0 first.  The override stays active."""
        feat = np.ascontiguousarray(np.asarray(feat, dtype=np.float64))
        out = np.zeros((feat.shape[1], self.height, self.width))
        for c0 in range(0, feat.shape[1], 3):
            n = self._override(feat, c0)
            out[c0:c0 + n] = self.forward()[0][:n]
        return out

    def backward_features(self, feat, dL_dF):
        """VJP of render_features: returns (grad_feat[N,C], dict of parameter gradients through alpha_k, T_k).
        Per pass the blend backward yields dL/df in g9[:,6:9]; the geometry gradients of the passes add up."""
        feat = np.ascontiguousarray(np.asarray(feat, dtype=np.float64))
        dL_dF = np.asarray(dL_dF, dtype=np.float64)
        gf = np.zeros_like(feat)
        total = None
        for c0 in range(0, feat.shape[1], 3):
            n = self._override(feat, c0)
            self.forward()
            g3 = np.zeros((3, self.height, self.width))
            g3[:n] = dL_dF[c0:c0 + n]
            g = self.backward(g3)
            gf[:, c0:c0 + n] = g["g9"][:, 6:6 + n]
            if total is None:
                total = {k: g[k].copy() for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")}
            else:
                for k in total:
                    total[k] += g[k]
        return gf, total

    def splat_flow(self, view, intr, dt_next):
        """Per-splat 2D displacement between the frames at t and t + dt_next: the conditional mean
        mu_xyz|t is linear in t (eq. 9), mu_c(t + d) = mu_c(t) + Sigma_1:3,4 / Sigma_44 d; both are projected with
        eq. 3 and subtracted.  Zero for primitives not visible at t or behind the camera at t + dt_next."""
        P = self.prims()
        V = np.asarray(view, dtype=np.float64).reshape(4, 4)
        fx, fy, cx, cy = intr
        flow = np.zeros((self.N, 2))
        for i in np.nonzero(P.status == STATUS_VISIBLE)[0]:
            _, Sigma = self.rot_cov(int(i))
            mu2 = P.mu_c[i] + Sigma[:3, 3] / Sigma[3, 3] * dt_next
            p2 = V[:3, :3] @ mu2 + V[:3, 3]
            if p2[2] <= 0:
                continue
            flow[i] = (fx * p2[0] / p2[2] + cx - P.uv[i, 0], fy * p2[1] / p2[2] + cy - P.uv[i, 1])
        return flow
