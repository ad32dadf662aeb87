"""Binding of the training-side entry points of include/fdgs.h (mask, regularisers, Adam, compact-model decode).

Marshalling only — every operation runs in the kernels of csrc/train.cu.  Tensors are torch CUDA tensors owned by the
caller; nothing here computes on the host and there is no fallback (fdgs.load() raises without the library).
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

from . import fdgs
from .fdgs import CAdamConfig, CCompactScene, CRegConfig, DeviceScene, FdgsError, _ptr, _stream, grads_struct

PARAMS = ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")


def mask_apply(mask_logit, mask_eps: float, opacity_logit, out=None):
    """eq. 21-23 forward: returns the opacity logits the renderer should see (-inf where M_hat = 0)."""
    import torch
    out = torch.empty_like(opacity_logit) if out is None else out
    rc = fdgs.load().fdgs_mask_apply(_ptr(mask_logit), float(mask_eps), _ptr(opacity_logit), _ptr(out),
                                     int(opacity_logit.numel()), _stream())
    if rc:
        raise FdgsError(rc, "fdgs_mask_apply")
    return out


def regularizers(ds: DeviceScene, grads: dict, lambda_sparse=0.0, lambda_covt=0.0, lambda_mask=0.0, mask_logit=None,
                 mask_eps=0.01, grad_mask_logit=None, losses=None):
    """eq. 24/26/27 fused forward + backward (+= into grads) and the mask's straight-through gradient.
    losses: float32[3] device tensor accumulated into (L_sparse, L_covt, L_mask), or None."""
    rc_ = CRegConfig(float(lambda_sparse), float(lambda_covt), float(lambda_mask), float(mask_eps))
    sc, g = ds.c_struct(), grads_struct(grads)
    rc = fdgs.load().fdgs_regularizers(C.byref(sc), _ptr(mask_logit), C.byref(rc_), C.byref(g), _ptr(grad_mask_logit),
                                       _ptr(losses), _stream())
    if rc:
        raise FdgsError(rc, "fdgs_regularizers")


def adam_step(param, grad, exp_avg, exp_avg_sq, step: int, lr: float, beta1=0.9, beta2=0.999, eps=1e-15, zero_grad=False):
    cfg = CAdamConfig(float(lr), float(beta1), float(beta2), float(eps), int(step))
    rc = fdgs.load().fdgs_adam_step(_ptr(param), _ptr(grad), _ptr(exp_avg), _ptr(exp_avg_sq), int(param.numel()),
                                    C.byref(cfg), 1 if zero_grad else 0, _stream())
    if rc:
        raise FdgsError(rc, "fdgs_adam_step")


class Adam:
    """Dense Adam over the six parameter arrays of a DeviceScene, one fdgs_adam_step launch per array
    (per-array learning rates as in [23]); state lives in HBM next to the parameters."""

    def __init__(self, ds: DeviceScene, lr: dict, beta1=0.9, beta2=0.999, eps=1e-15):
        import torch
        self.ds, self.lr, self.b1, self.b2, self.eps, self.t = ds, dict(lr), beta1, beta2, eps, 0
        self.m = {k: torch.zeros_like(getattr(ds, k)) for k in PARAMS}
        self.v = {k: torch.zeros_like(getattr(ds, k)) for k in PARAMS}

    def step(self, grads: dict, zero_grad=True):
        self.t += 1
        for k in PARAMS:
            adam_step(getattr(self.ds, k), grads[k], self.m[k], self.v[k], self.t, self.lr[k], self.b1, self.b2, self.eps,
                      zero_grad)


def decode_compact(c: dict, sh_degree: int, n_time: int, out: Optional[DeviceScene] = None) -> DeviceScene:
    """c: dict of CUDA tensors — mean_f16 [N,4] float16, opacity_code [N] uint8, opacity_lo/hi floats, scale_idx,
    rot_l_idx, rot_r_idx, dc_idx, rest_idx [N,stages] uint8, scale_cb / rot_cb [stages,entries,4], dc_cb [stages,entries,3],
    rest_cb [stages,entries,(K-1)*3] float32.  Returns (or fills) a DeviceScene."""
    import torch
    N = int(c["mean_f16"].shape[0])
    K = n_time * (sh_degree + 1) ** 2
    dev = c["mean_f16"].device
    if out is None:
        e = lambda *s: torch.empty(s, dtype=torch.float32, device=dev)
        out = DeviceScene(sh_degree, n_time, e(N, 4), e(N, 4), e(N, 4), e(N, 4), e(N), e(N, K, 3))
    cs = CCompactScene()
    cs.N, cs.sh_degree, cs.n_time = N, sh_degree, n_time
    cs.mean_f16, cs.opacity_code = _ptr(c["mean_f16"]), _ptr(c["opacity_code"])
    cs.opacity_lo, cs.opacity_hi, cs.opacity_bits = float(c["opacity_lo"]), float(c["opacity_hi"]), int(c.get("opacity_bits", 8))
    for name, idx in (("scale", "scale_idx"), ("dc", "dc_idx"), ("rest", "rest_idx")):
        cb = c.get(name + "_cb")
        if cb is None:
            continue
        setattr(cs, name + "_stages", int(cb.shape[0]))
        setattr(cs, name + "_entries", int(cb.shape[1]))
        setattr(cs, idx, _ptr(c[idx]))
        setattr(cs, name + "_cb", _ptr(cb))
    cs.rot_stages, cs.rot_entries = int(c["rot_cb"].shape[0]), int(c["rot_cb"].shape[1])
    cs.rot_l_idx, cs.rot_r_idx, cs.rot_cb = _ptr(c["rot_l_idx"]), _ptr(c["rot_r_idx"]), _ptr(c["rot_cb"])
    sc = out.c_struct()
    rc = fdgs.load().fdgs_decode_compact(C.byref(cs), C.byref(sc), _stream())
    if rc:
        raise FdgsError(rc, "fdgs_decode_compact")
    return out
