"""torch.autograd front end over the C-ABI renderer: ``render(params, view)`` returns the image (optionally depth and
accumulated opacity) as differentiable tensors; backward runs fdgs_render_backward(_aux).  Marshalling only: every step of
the path runs in the CUDA kernels of libfdgs.so (there is no CPU fallback).

    params = {k: torch.nn.Parameter(...) for k in ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")}
    rast = Rasterizer(sh_degree=3, n_time=3, width=W, height=H, pair_capacity=16 << 20)
    image = rast(params, view)                       # [3,H,W]
    image, depth, opacity = rast(params, view, aux=True)
    loss.backward()                                  # gradients land in params[k].grad

One Rasterizer owns one workspace: a second forward overwrites the state the backward of the first one needs (render,
backward, render, backward ...; use one Rasterizer per view of a batch to keep several graphs alive).
"""
from __future__ import annotations

import torch

from . import fdgs

PARAM_KEYS = ("mean", "log_scale", "quat_l", "quat_r", "opacity_logit", "sh")


class _Render(torch.autograd.Function):
    @staticmethod
    def forward(ctx, rast, cview, aux, mean, log_scale, quat_l, quat_r, opacity_logit, sh):
        tensors = [mean, log_scale, quat_l, quat_r, opacity_logit, sh]
        for t in tensors:
            if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
                raise ValueError("parameters must be contiguous float32 CUDA tensors")
        ds = fdgs.DeviceScene(rast.sh_degree, rast.n_time, *[t.detach() for t in tensors])
        if ds.K * 3 != sh.shape[1] * sh.shape[2] or sh.shape[0] != ds.N:
            raise ValueError(f"sh must be [N, {ds.K}, 3]")
        r = rast._renderer(ds)
        r.preprocess(cview, sync=True)      # raises FdgsError(ERR_PAIR_OVERFLOW) instead of training on a background image
        if aux:
            r.forward_aux(cview)
        else:
            r.forward(cview)
        ctx.rast, ctx.cview, ctx.aux, ctx.ds = rast, cview, aux, ds
        rast._generation += 1
        ctx.generation = rast._generation
        image = r.image.clone()
        if not aux:
            return image
        return image, r.depth_map.clone(), 1.0 - r.final_T

    @staticmethod
    def backward(ctx, g_image, g_depth=None, g_opacity=None):
        rast, r = ctx.rast, ctx.rast._r
        if ctx.generation != rast._generation:
            raise RuntimeError("this Rasterizer has rendered again since: its workspace no longer holds this forward "
                               "(use one Rasterizer per graph kept alive)")
        grads = ctx.ds.zero_grads()
        g_image = g_image.contiguous().float() if g_image is not None else torch.zeros_like(r.image)
        if ctx.aux:
            gd = g_depth.contiguous().float() if g_depth is not None else None
            go = g_opacity.contiguous().float() if g_opacity is not None else None
            r.backward_aux(ctx.cview, g_image, gd, go, grads)
        else:
            r.backward(ctx.cview, g_image, grads)
        return (None, None, None) + tuple(grads[k] for k in PARAM_KEYS)


class Rasterizer:
    """Differentiable renderer for scenes of a fixed size class (N is taken from the parameters at each call)."""

    def __init__(self, sh_degree: int, n_time: int, width: int, height: int, pair_capacity: int, cfg=None):
        self.sh_degree, self.n_time = int(sh_degree), int(n_time)
        self.width, self.height, self.cap, self.cfg = int(width), int(height), int(pair_capacity), cfg
        self._r, self._n, self._generation = None, -1, 0

    def _renderer(self, ds):
        if self._r is None or self._n != ds.N:
            self._r, self._n = fdgs.Renderer(ds, self.width, self.height, self.cap, self.cfg), ds.N
        else:
            self._r.ds, self._r._cs = ds, ds.c_struct()
        return self._r

    def __call__(self, params: dict, view, aux: bool = False):
        cview = view if isinstance(view, fdgs.CView) else fdgs.make_view(view)
        return _Render.apply(self, cview, bool(aux), *[params[k] for k in PARAM_KEYS])
