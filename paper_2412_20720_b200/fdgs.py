"""Thin ctypes binding over the C-ABI library of include/fdgs.h — argument marshalling only.

Every step of the path runs in the hand-written CUDA kernels of libfdgs.so; PyTorch is used for
device memory and streams.  There is NO CPU fallback: the first call raises if the library has not
been built (``python -m paper_2412_20720_b200.build``) or if no CUDA device is present.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdgs.so")
_lib = None

OK, ERR_INVALID, ERR_WORKSPACE, ERR_CUDA, ERR_PAIR_OVERFLOW, ERR_STATIC_LIMIT = 0, -1, -2, -3, -4, -5
STATIC_WS_BYTES = 8 << 20
(EXPORT_STATUS, EXPORT_RECORDS, EXPORT_RECTS, EXPORT_TILES_TOUCHED, _EXPORT_UNUSED_4, EXPORT_SORTED_KEYS,
 EXPORT_SORTED_VALS, EXPORT_RANGES, EXPORT_SPLAT_GRADS, EXPORT_DEPTH_ORDER, EXPORT_SPLAT_GRAD_DEPTH) = range(11)

EXPORTED_SYMBOLS = ["fdgs_default_config", "fdgs_workspace_bytes", "fdgs_preprocess", "fdgs_render_forward",
                    "fdgs_render_backward", "fdgs_l1_loss", "fdgs_step_host", "fdgs_debug_export",
                    "fdgs_launch_count", "fdgs_strerror", "fdgs_set_stage_timing", "fdgs_get_stage_ms",
                    "fdgs_debug_blend_stats", "fdgs_step_batch", "fdgs_debug_cull_status", "fdgs_render_forward_aux",
                    "fdgs_render_backward_aux", "fdgs_debug_measure_peaks", "fdgs_mask_apply", "fdgs_regularizers",
                    "fdgs_adam_step", "fdgs_decode_compact", "fdgs_features_scratch_bytes", "fdgs_render_features_forward",
                    "fdgs_render_features_backward", "fdgs_splat_flow", "fdgs_render_forward_static"]
MAX_BATCH = 8


class CScene(C.Structure):
    _fields_ = [("N", C.c_int32), ("sh_degree", C.c_int32), ("n_time", C.c_int32), ("mean", C.c_void_p),
                ("log_scale", C.c_void_p), ("quat_l", C.c_void_p), ("quat_r", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("sh", C.c_void_p)]


class CView(C.Structure):
    _fields_ = [("view", C.c_float * 16), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("width", C.c_int32), ("height", C.c_int32), ("t", C.c_float), ("period_T", C.c_float),
                ("bg", C.c_float * 3)]


class CConfig(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("marginal_min", "alpha_min", "alpha_max", "transmittance_min", "dilation",
                                         "cutoff_sigma", "znear", "guard")]


class CGrads(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh", "mean2d", "densify")]


class CViewBuffers(C.Structure):
    _fields_ = [("ws", C.c_void_p), ("ws_bytes", C.c_size_t), ("target_host", C.c_void_p), ("target_dev", C.c_void_p),
                ("image", C.c_void_p), ("final_T", C.c_void_p), ("n_contrib", C.c_void_p), ("dL_dimage", C.c_void_p)]


class CRegConfig(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("lambda_sparse", "lambda_covt", "lambda_mask", "mask_eps")]


class CAdamConfig(C.Structure):
    _fields_ = [("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_int32)]


class CCompactScene(C.Structure):
    _fields_ = [("N", C.c_int32), ("sh_degree", C.c_int32), ("n_time", C.c_int32), ("mean_f16", C.c_void_p),
                ("opacity_code", C.c_void_p), ("opacity_lo", C.c_float), ("opacity_hi", C.c_float), ("opacity_bits", C.c_int32),
                ("scale_stages", C.c_int32), ("scale_entries", C.c_int32), ("scale_idx", C.c_void_p), ("scale_cb", C.c_void_p),
                ("rot_stages", C.c_int32), ("rot_entries", C.c_int32), ("rot_l_idx", C.c_void_p), ("rot_r_idx", C.c_void_p),
                ("rot_cb", C.c_void_p),
                ("dc_stages", C.c_int32), ("dc_entries", C.c_int32), ("dc_idx", C.c_void_p), ("dc_cb", C.c_void_p),
                ("rest_stages", C.c_int32), ("rest_entries", C.c_int32), ("rest_idx", C.c_void_p), ("rest_cb", C.c_void_p)]


class FdgsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})")


def load():
    """Loads libfdgs.so; raises loudly if it is missing (the product has no fallback path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build the CUDA library first "
                           "(python -m paper_2412_20720_b200.build); there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    vp, sz, i64, i32 = C.c_void_p, C.c_size_t, C.c_int64, C.c_int32
    lib.fdgs_default_config.argtypes = [C.POINTER(CConfig)]
    lib.fdgs_workspace_bytes.argtypes = [i32, i32, i32, i32, i64, C.POINTER(sz)]
    lib.fdgs_preprocess.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp,
                                    C.POINTER(i64), C.POINTER(i32)]
    lib.fdgs_render_forward.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, vp, vp]
    lib.fdgs_render_backward.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, vp,
                                         vp, C.POINTER(CGrads)]
    lib.fdgs_render_forward_aux.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, vp, vp, vp]
    lib.fdgs_render_backward_aux.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, vp, vp,
                                             vp, vp, C.POINTER(CGrads)]
    lib.fdgs_l1_loss.argtypes = [vp, vp, i64, vp, vp, vp]
    lib.fdgs_step_host.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, vp, vp, vp,
                                   vp, vp, vp, C.POINTER(CGrads), vp]
    lib.fdgs_step_batch.argtypes = [C.POINTER(CScene), C.POINTER(CView), i32, C.POINTER(CConfig), i64, C.POINTER(CViewBuffers), vp, vp,
                                    C.POINTER(CGrads), vp, i32]
    lib.fdgs_debug_cull_status.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, vp]
    lib.fdgs_debug_measure_peaks.argtypes = [vp, sz, vp, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    lib.fdgs_debug_export.argtypes = [vp, sz, C.c_int, vp, sz, vp]
    lib.fdgs_set_stage_timing.argtypes = [C.c_int]
    lib.fdgs_get_stage_ms.argtypes = [C.POINTER(C.c_float)]
    lib.fdgs_debug_blend_stats.argtypes = [C.POINTER(CView), C.POINTER(CConfig), vp, sz, i32, i32, i64, vp, vp]
    lib.fdgs_mask_apply.argtypes = [vp, C.c_float, vp, vp, i32, vp]
    lib.fdgs_regularizers.argtypes = [C.POINTER(CScene), vp, C.POINTER(CRegConfig), C.POINTER(CGrads), vp, vp, vp]
    lib.fdgs_adam_step.argtypes = [vp, vp, vp, vp, i64, C.POINTER(CAdamConfig), i32, vp]
    lib.fdgs_decode_compact.argtypes = [C.POINTER(CCompactScene), C.POINTER(CScene), vp]
    lib.fdgs_features_scratch_bytes.argtypes = [i32, i32, i32, C.POINTER(sz)]
    lib.fdgs_render_features_forward.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, i32,
                                                 vp, sz, vp]
    lib.fdgs_render_features_backward.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, vp, i32,
                                                  vp, sz, vp, vp, vp, vp, C.POINTER(CGrads)]
    lib.fdgs_splat_flow.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), vp, sz, i64, vp, C.c_float, vp]
    lib.fdgs_render_forward_static.argtypes = [C.POINTER(CScene), C.POINTER(CView), C.POINTER(CConfig), i64, vp, vp, vp, vp, vp]
    lib.fdgs_launch_count.restype = i64
    lib.fdgs_strerror.restype = C.c_char_p
    lib.fdgs_strerror.argtypes = [C.c_int]
    for name in EXPORTED_SYMBOLS:
        if name not in ("fdgs_launch_count", "fdgs_strerror"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load().fdgs_strerror(int(code)).decode()


def launch_count() -> int:
    return int(load().fdgs_launch_count())


# "colour_side_stream": the colour kernel that fdgs_render_forward runs next to the depth sort and the row scatter (degree 3)
STAGES = ("preprocess", "compact+tile_grid", "sort_depth", "tile_lists", "blend_fwd", "blend_bwd", "preprocess_bwd", "colour_side_stream")


def set_stage_timing(on: bool):
    rc = load().fdgs_set_stage_timing(1 if on else 0)
    if rc:
        raise FdgsError(rc, "fdgs_set_stage_timing")


def stage_ms() -> dict:
    buf = (C.c_float * 8)()
    rc = load().fdgs_get_stage_ms(buf)
    if rc:
        raise FdgsError(rc, "fdgs_get_stage_ms")
    return {k: float(buf[i]) for i, k in enumerate(STAGES)}


def measure_peaks() -> dict:
    """Measured FP32-FMA issue peak (T lane-instructions/s) and MUFU.EX2 peak (T/s) of the current device."""
    import torch
    scratch = torch.empty(4 * 8 * 256 * 256, dtype=torch.uint8, device="cuda")
    a, b = C.c_float(0), C.c_float(0)
    rc = load().fdgs_debug_measure_peaks(scratch.data_ptr(), scratch.numel(), _stream(), C.byref(a), C.byref(b))
    if rc:
        raise FdgsError(rc, "fdgs_debug_measure_peaks")
    return {"fma_tlane_per_s": float(a.value), "mufu_ex2_t_per_s": float(b.value)}


def default_config(**overrides) -> CConfig:
    cfg = CConfig()
    rc = load().fdgs_default_config(C.byref(cfg))
    if rc:
        raise FdgsError(rc, "fdgs_default_config")
    for k, v in overrides.items():
        if k == "full_support":
            continue
        setattr(cfg, k, float(v))
    return cfg


def make_view(view) -> CView:
    """From a scenes.View (or anything with the same attributes)."""
    import numpy as np
    cv = CView()
    flat = np.asarray(view.view, dtype=np.float32).reshape(16)
    for i in range(16):
        cv.view[i] = float(flat[i])
    cv.fx, cv.fy, cv.cx, cv.cy = float(view.fx), float(view.fy), float(view.cx), float(view.cy)
    cv.width, cv.height, cv.t, cv.period_T = int(view.width), int(view.height), float(view.t), float(view.period_T)
    for i in range(3):
        cv.bg[i] = float(view.bg[i])
    return cv


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream() -> int:
    import torch
    return torch.cuda.current_stream().cuda_stream


@dataclass
class DeviceScene:
    """The six parameter arrays resident in HBM (torch float32 CUDA tensors)."""
    sh_degree: int
    n_time: int
    mean: "torch.Tensor"
    log_scale: "torch.Tensor"
    quat_l: "torch.Tensor"
    quat_r: "torch.Tensor"
    opacity_logit: "torch.Tensor"
    sh: "torch.Tensor"

    @property
    def N(self):
        return int(self.mean.shape[0])

    @property
    def K(self):
        return self.n_time * (self.sh_degree + 1) ** 2

    @classmethod
    def from_scene(cls, scene, device="cuda:0"):
        import torch
        f = lambda a: torch.from_numpy(a.astype("float32", copy=False)).contiguous().to(device)
        return cls(scene.sh_degree, scene.n_time, f(scene.mean), f(scene.log_scale), f(scene.quat_l), f(scene.quat_r),
                   f(scene.opacity_logit), f(scene.sh))

    def c_struct(self) -> CScene:
        return CScene(self.N, self.sh_degree, self.n_time, _ptr(self.mean), _ptr(self.log_scale), _ptr(self.quat_l),
                      _ptr(self.quat_r), _ptr(self.opacity_logit), _ptr(self.sh))

    def zero_grads(self, with_mean2d=False, with_densify=False):
        import torch
        g = {k: torch.zeros_like(getattr(self, k)) for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")}
        g["mean2d"] = torch.zeros((self.N, 2), device=self.mean.device) if with_mean2d else None
        g["densify"] = torch.zeros((self.N, 3), device=self.mean.device) if with_densify else None
        return g


def grads_struct(g: dict) -> CGrads:
    return CGrads(_ptr(g["mean"]), _ptr(g["log_scale"]), _ptr(g["quat_l"]), _ptr(g["quat_r"]), _ptr(g["opacity_logit"]),
                  _ptr(g["sh"]), _ptr(g.get("mean2d")), _ptr(g.get("densify")))


def render_forward_static(dscene: "DeviceScene", cview: CView, pair_capacity: int, image, final_T, n_contrib,
                          overflow=None, cfg: Optional[CConfig] = None) -> None:
    """fdgs_render_forward_static: forward of one view on the workspace built into the library (no allocation).

    image [3,H,W] f32, final_T [H,W] f32, n_contrib [H,W] i32, overflow (optional) [1] i32: caller-owned CUDA tensors.
    Raises FdgsError(ERR_STATIC_LIMIT) if workspace_bytes(...) > STATIC_WS_BYTES.  Asynchronous on the current stream."""
    cs = dscene.c_struct()
    cfg = cfg if cfg is not None else default_config()
    rc = load().fdgs_render_forward_static(C.byref(cs), C.byref(cview), C.byref(cfg), int(pair_capacity), _stream(),
                                           image.data_ptr(), final_T.data_ptr(), n_contrib.data_ptr(), _ptr(overflow))
    if rc:
        raise FdgsError(rc, "fdgs_render_forward_static")


def workspace_bytes(N, K, width, height, pair_capacity) -> int:
    out = C.c_size_t(0)
    rc = load().fdgs_workspace_bytes(int(N), int(K), int(width), int(height), int(pair_capacity), C.byref(out))
    if rc:
        raise FdgsError(rc, "fdgs_workspace_bytes")
    return int(out.value)


class Renderer:
    """Owns the workspace and output buffers for one (scene size, resolution, pair capacity)."""

    def __init__(self, dscene: DeviceScene, width: int, height: int, pair_capacity: int, cfg: Optional[CConfig] = None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("fdgs needs a CUDA device (sm_100a); there is no CPU fallback")
        self.lib = load()
        self.ds, self.width, self.height, self.cap = dscene, int(width), int(height), int(pair_capacity)
        self.cfg = cfg if cfg is not None else default_config()
        dev = dscene.mean.device
        self.ws_bytes = workspace_bytes(dscene.N, dscene.K, width, height, pair_capacity)
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=dev)
        self.image = torch.empty((3, height, width), dtype=torch.float32, device=dev)
        self.final_T = torch.empty((height, width), dtype=torch.float32, device=dev)
        self.n_contrib = torch.empty((height, width), dtype=torch.int32, device=dev)
        self.dL_dimage = torch.empty((3, height, width), dtype=torch.float32, device=dev)
        self.loss = torch.zeros(1, dtype=torch.float32, device=dev)
        self.target_dev = torch.empty((3, height, width), dtype=torch.float32, device=dev)
        self._cs = dscene.c_struct()

    # -- the three calls of the boundary ---------------------------------------------------------
    def preprocess(self, cview: CView, sync: bool = False):
        npairs, nvis = C.c_int64(-1), C.c_int32(-1)
        rc = self.lib.fdgs_preprocess(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(), self.ws_bytes,
                                      self.cap, _stream(), C.byref(npairs) if sync else None, C.byref(nvis) if sync else None)
        if rc:
            raise FdgsError(rc, "fdgs_preprocess")
        return (int(npairs.value), int(nvis.value)) if sync else None

    def forward(self, cview: CView):
        rc = self.lib.fdgs_render_forward(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(),
                                          self.ws_bytes, self.cap, _stream(), self.image.data_ptr(), self.final_T.data_ptr(),
                                          self.n_contrib.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_render_forward")
        return self.image

    def backward(self, cview: CView, dL_dimage, grads: dict):
        cg = grads_struct(grads)
        rc = self.lib.fdgs_render_backward(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(),
                                           self.ws_bytes, self.cap, _stream(), dL_dimage.data_ptr(), self.final_T.data_ptr(),
                                           self.n_contrib.data_ptr(), C.byref(cg))
        if rc:
            raise FdgsError(rc, "fdgs_render_backward")

    def forward_aux(self, cview: CView):
        """Forward with the auxiliary depth channel: returns (image, depth_map); opacity is 1 - self.final_T."""
        import torch
        if getattr(self, "depth_map", None) is None:
            self.depth_map = torch.empty((self.height, self.width), dtype=torch.float32, device=self.ws.device)
        rc = self.lib.fdgs_render_forward_aux(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(),
                                              self.ws_bytes, self.cap, _stream(), self.image.data_ptr(), self.final_T.data_ptr(),
                                              self.n_contrib.data_ptr(), self.depth_map.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_render_forward_aux")
        return self.image, self.depth_map

    def backward_aux(self, cview: CView, dL_dimage, dL_ddepth, dL_dopacity, grads: dict):
        cg = grads_struct(grads)
        rc = self.lib.fdgs_render_backward_aux(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(),
                                               self.ws_bytes, self.cap, _stream(), dL_dimage.data_ptr(), _ptr(dL_ddepth),
                                               _ptr(dL_dopacity), self.final_T.data_ptr(), self.n_contrib.data_ptr(), C.byref(cg))
        if rc:
            raise FdgsError(rc, "fdgs_render_backward_aux")

    # ---- feature channels / optical flow (include/fdgs.h "Feature channels") ----
    def _feat_scratch(self):
        import torch
        if getattr(self, "_fscratch", None) is None:
            n = C.c_size_t(0)
            rc = self.lib.fdgs_features_scratch_bytes(self.ds.N, self.width, self.height, C.byref(n))
            if rc:
                raise FdgsError(rc, "fdgs_features_scratch_bytes")
            self._fscratch = torch.empty(int(n.value), dtype=torch.uint8, device=self.ws.device)
        return self._fscratch

    def features_forward(self, cview: CView, feat, out=None):
        """feat [N,C] float32 CUDA -> [C,H,W]; call after preprocess + forward of this view."""
        import torch
        Cn = int(feat.shape[1])
        out = torch.empty((Cn, self.height, self.width), dtype=torch.float32, device=feat.device) if out is None else out
        sc = self._feat_scratch()
        rc = self.lib.fdgs_render_features_forward(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(),
                                                   self.ws_bytes, self.cap, _stream(), feat.data_ptr(), Cn, sc.data_ptr(),
                                                   sc.numel(), out.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_render_features_forward")
        return out

    def features_backward(self, cview: CView, feat, dL_dout, grad_feat, grads: Optional[dict] = None):
        Cn = int(feat.shape[1])
        sc = self._feat_scratch()
        cg = grads_struct(grads) if grads is not None else None
        rc = self.lib.fdgs_render_features_backward(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(),
                                                    self.ws_bytes, self.cap, _stream(), feat.data_ptr(), Cn, sc.data_ptr(),
                                                    sc.numel(), dL_dout.data_ptr(), self.final_T.data_ptr(),
                                                    self.n_contrib.data_ptr(), grad_feat.data_ptr(),
                                                    C.byref(cg) if cg is not None else None)
        if rc:
            raise FdgsError(rc, "fdgs_render_features_backward")

    def splat_flow(self, cview: CView, dt_next: float):
        """Per-splat 2D displacement [N,2] between t and t + dt_next; call after preprocess."""
        import torch
        flow = torch.empty((self.ds.N, 2), dtype=torch.float32, device=self.ws.device)
        rc = self.lib.fdgs_splat_flow(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(), self.ws_bytes,
                                      self.cap, _stream(), float(dt_next), flow.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_splat_flow")
        return flow

    def l1_loss(self, target):
        """loss += mean|image - target|; writes self.dL_dimage."""
        rc = self.lib.fdgs_l1_loss(self.image.data_ptr(), target.data_ptr(), self.image.numel(), self.dL_dimage.data_ptr(),
                                   self.loss.data_ptr(), _stream())
        if rc:
            raise FdgsError(rc, "fdgs_l1_loss")

    def step_host(self, cview: CView, target_host, result_host, grads: Optional[dict]):
        """One view end to end with HOST target / result buffers (fdgs_step_host)."""
        cg = grads_struct(grads) if grads is not None else None
        rc = self.lib.fdgs_step_host(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(), self.ws_bytes,
                                     self.cap, _stream(), _ptr(target_host), self.target_dev.data_ptr(), self.image.data_ptr(),
                                     self.final_T.data_ptr(), self.n_contrib.data_ptr(), self.dL_dimage.data_ptr(),
                                     self.loss.data_ptr(), C.byref(cg) if cg is not None else None, result_host.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_step_host")

    # -- measurement hooks -----------------------------------------------------------------------
    def blend_stats(self, cview: CView):
        """(pairs walked, pairs reaching exp2, pairs composited, splats staged) of the last forward on this workspace."""
        import torch
        out = torch.zeros(4, dtype=torch.int64, device=self.ws.device)
        rc = self.lib.fdgs_debug_blend_stats(C.byref(cview), C.byref(self.cfg), self.ws.data_ptr(), self.ws_bytes, self.ds.N,
                                             self.ds.K, self.cap, _stream(), out.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_debug_blend_stats")
        return [int(x) for x in out.cpu()]

    def cull_status(self, cview: CView):
        """uint8[N]: 0 visible, 1 temporal marginal, 2 near plane, 3 empty rectangle, 4 non-finite."""
        import torch
        out = torch.zeros(max(self.ds.N, 1), dtype=torch.uint8, device=self.ws.device)
        rc = self.lib.fdgs_debug_cull_status(C.byref(self._cs), C.byref(cview), C.byref(self.cfg), _stream(), out.data_ptr())
        if rc:
            raise FdgsError(rc, "fdgs_debug_cull_status")
        return out[:self.ds.N]

    # -- parity hooks -----------------------------------------------------------------------------
    def export(self, what: int):
        import torch
        dev = self.ws.device
        N, tiles = self.ds.N, ((self.width + 15) // 16) * ((self.height + 15) // 16)
        status = torch.zeros(4, dtype=torch.int64, device=dev)
        rc = self.lib.fdgs_debug_export(self.ws.data_ptr(), self.ws_bytes, EXPORT_STATUS, status.data_ptr(), 32, _stream())
        if rc not in (OK, ERR_PAIR_OVERFLOW):
            raise FdgsError(rc, "fdgs_debug_export(status)")
        D, nvis, overflow = int(status[0]), int(status[1]), int(status[2])
        if what == EXPORT_STATUS:
            return dict(num_pairs=D, num_visible=nvis, overflow=overflow, pair_capacity=int(status[3]))
        if overflow:
            D = 0
        shapes = {EXPORT_RECORDS: ((N, 12), torch.float32), EXPORT_RECTS: ((N, 4), torch.int32),
                  EXPORT_TILES_TOUCHED: ((N,), torch.int32),
                  EXPORT_SORTED_KEYS: ((D,), torch.int64), EXPORT_SORTED_VALS: ((D,), torch.int32),
                  EXPORT_RANGES: ((tiles, 2), torch.int32), EXPORT_SPLAT_GRADS: ((N, 9), torch.float32),
                  EXPORT_DEPTH_ORDER: ((nvis,), torch.int32), EXPORT_SPLAT_GRAD_DEPTH: ((N,), torch.float32)}
        shape, dt = shapes[what]
        out = torch.zeros(shape, dtype=dt, device=dev)
        if out.numel() == 0:
            return out
        rc = self.lib.fdgs_debug_export(self.ws.data_ptr(), self.ws_bytes, what, out.data_ptr(), out.numel() * out.element_size(),
                                        _stream())
        if rc:
            raise FdgsError(rc, f"fdgs_debug_export({what})")
        return out


class BatchStep:
    """One optimisation step over a batch of views through fdgs_step_batch: one Renderer (workspace + buffers) per view."""

    def __init__(self, dscene: DeviceScene, width: int, height: int, pair_capacity: int, num_views: int, cfg: Optional[CConfig] = None):
        import torch
        if not 1 <= num_views <= MAX_BATCH:
            raise ValueError(f"num_views must be in 1..{MAX_BATCH}")
        self.lib = load()
        self.ds, self.cap, self.num_views = dscene, int(pair_capacity), int(num_views)
        self.renderers = [Renderer(dscene, width, height, pair_capacity, cfg) for _ in range(num_views)]
        self.cfg = self.renderers[0].cfg
        self.loss = torch.zeros(num_views, dtype=torch.float32, device=dscene.mean.device)
        self._cs = dscene.c_struct()

    def step(self, cviews, grads: dict, targets_host=None, loss_host=None, zero_grads=False):
        """targets_host: list of pinned [3,H,W] host tensors (copied inside the call) or None if every renderer's
        target_dev already holds its target.  loss_host: pinned float tensor [num_views] (copied back, synchronises)
        or None (asynchronous).  zero_grads: the library zeroes the gradient arrays itself (FDGS_STEP_ZERO_GRADS)."""
        n = self.num_views
        views = (CView * n)(*cviews)
        bufs = (CViewBuffers * n)()
        for i, r in enumerate(self.renderers):
            bufs[i] = CViewBuffers(r.ws.data_ptr(), r.ws_bytes, _ptr(targets_host[i]) if targets_host is not None else None,
                                   r.target_dev.data_ptr(), r.image.data_ptr(), r.final_T.data_ptr(), r.n_contrib.data_ptr(),
                                   r.dL_dimage.data_ptr())
        cg = grads_struct(grads)
        rc = self.lib.fdgs_step_batch(C.byref(self._cs), views, n, C.byref(self.cfg), self.cap, bufs, _stream(), self.loss.data_ptr(),
                                      C.byref(cg), _ptr(loss_host), 1 if zero_grads else 0)
        if rc:
            raise FdgsError(rc, "fdgs_step_batch")
