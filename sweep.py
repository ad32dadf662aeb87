"""Secondary measurements of BASELINE.json's configs 2, 4 and 5 (bench.py times the headline config 3).

    python sweep.py [--frames 120] [--max-n 8000000] [--skip-train] [--train-terms]

cfg5: forward-only render throughput over Gaussian count x resolution at evenly spaced query times: FPS (one frame at a
time), per-stage ms (preprocess / sort incl. compaction, duplication and ranges / blend) and the fraction culled by the
marginal temporal weight.  cfg2 / cfg4: forward+backward steps/s of their batch through fdgs_step_batch.
One JSON line per measurement on stdout.  Synthetic seeded scenes (scenes.py); no CPU fallback.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import numpy as np


ONCE = False      # --once: every operation runs twice (1 warm-up + 1 timed) so that a profiler capture covers all kernels


def _timed(fn, iters, warm, flush):
    import torch
    if ONCE:
        iters, warm = 1, 1
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    tot = 0.0
    for _ in range(iters):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        tot += e0.elapsed_time(e1)
    return tot / iters


def sweep_cfg5(frames, max_n, flush):
    import torch
    from paper_2412_20720_b200 import fdgs, scenes
    for (w, h) in ((1352, 1014), (1920, 1080)):
        for n in (100_000, 500_000, 1_000_000, 2_000_000, 4_000_000, 8_000_000):
            if n > max_n:
                continue
            sc = scenes.sweep(N=n, width=w, height=h, n_frames=120)
            ds = fdgs.DeviceScene.from_scene(sc)
            cap = max(1 << 22, 16 * n)
            r = fdgs.Renderer(ds, w, h, cap)
            idx = np.linspace(0, 119, frames).round().astype(int)
            cvs = [fdgs.make_view(sc.views[i]) for i in idx]
            ms, culled, pairs, nvis = [], [], [], []
            fdgs.set_stage_timing(True)
            stage = {k: 0.0 for k in fdgs.STAGES[:5] + ("colour_side_stream",)}
            for cv in cvs:
                def frame():
                    r.preprocess(cv)
                    r.forward(cv)
                ms.append(_timed(frame, 3, 2, flush))
                for k, v in fdgs.stage_ms().items():
                    if k in stage:
                        stage[k] += v / len(cvs)
                st = r.export(fdgs.EXPORT_STATUS)
                if st["overflow"]:
                    raise RuntimeError(f"pair capacity exceeded: {st}")
                culled.append(float((r.cull_status(cv) == 1).sum().item()) / n)     # culled by the marginal temporal weight
                pairs.append(st["num_pairs"]); nvis.append(st["num_visible"])
            fdgs.set_stage_timing(False)
            ms_frame = float(np.mean(ms))
            print(json.dumps({"config": "cfg5_sweep", "N": n, "width": w, "height": h, "frames": len(cvs), "fps": 1e3 / ms_frame,
                              "ms_per_frame": ms_frame, "ms_min": float(np.min(ms)), "ms_max": float(np.max(ms)),
                              # "preprocess": the geometry kernel on the critical path; the colour of the survivors runs on the
                              # side stream of fdgs_render_forward UNDER the sort stage (its own time is reported next to it)
                              "stage_ms": {"preprocess": stage["preprocess"],
                                           "sort": stage["compact+tile_grid"] + stage["sort_depth"] + stage["tile_lists"],
                                           "blend": stage["blend_fwd"], "colour_under_sort": stage["colour_side_stream"]},
                              "culled_by_marginal_fraction": float(np.mean(culled)), "visible_mean": float(np.mean(nvis)),
                              "pairs_mean": float(np.mean(pairs))}), flush=True)
            del r, ds, sc
            torch.cuda.empty_cache()


def train_cfg(name, scene, cap, flush):
    import torch
    from paper_2412_20720_b200 import fdgs, scenes
    ds = fdgs.DeviceScene.from_scene(scene)
    v0 = scene.views[0]
    nv = len(scene.views)
    bs = fdgs.BatchStep(ds, v0.width, v0.height, cap, nv)
    cvs = [fdgs.make_view(v) for v in scene.views]
    for i, rr in enumerate(bs.renderers):
        rr.target_dev.copy_(torch.from_numpy(scenes.target_image(scene.seed, i, v0.width, v0.height)).cuda())
    grads = ds.zero_grads()

    def step():
        for g in grads.values():
            if g is not None:
                g.zero_()
        bs.step(cvs, grads)
    ms = _timed(step, 5, 3, flush)
    sts = [rr.export(fdgs.EXPORT_STATUS) for rr in bs.renderers]
    if any(s["overflow"] for s in sts):
        raise RuntimeError(f"pair capacity exceeded: {sts}")
    print(json.dumps({"config": name, "N": scene.N, "width": v0.width, "height": v0.height, "views_per_step": nv,
                      "steps_per_s": 1e3 / ms, "ms_per_step": ms, "pairs_per_view": [s["num_pairs"] for s in sts],
                      "visible_per_view": [s["num_visible"] for s in sts], "loss": float(bs.loss.sum())}), flush=True)


def train_terms(flush, n=1_000_000):
    """SURVEY 8(f) f2-f4 kernels at cfg3's size (N = 1 M, K = 48): ms and achieved HBM GB/s on ALGORITHMIC bytes
    (DESIGN.md section 10): regularisers 176 B/primitive, Adam 28 B/element (32 with zero_grad) over the 161 floats of a
    primitive, decode 41 B read + 644 B written per primitive."""
    import torch
    from paper_2412_20720_b200 import fdgs, scenes, train
    sc = scenes.multiview_video(N=n, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    g = ds.zero_grads()
    m = torch.randn(n, device="cuda")
    gm, losses = torch.zeros(n, device="cuda"), torch.zeros(3, device="cuda")
    ms = _timed(lambda: train.regularizers(ds, g, 0.01, 0.01, 0.01, m, 0.01, gm, losses), 20, 5, flush)
    out = {"config": "train_terms", "N": n, "K": ds.K,
           "regularizers": {"ms": ms, "bytes": 176 * n, "GBps": 176 * n / ms / 1e6}}
    ms = _timed(lambda: train.mask_apply(m, 0.01, ds.opacity_logit, gm), 20, 5, flush)
    out["mask_apply"] = {"ms": ms, "bytes": 12 * n, "GBps": 12 * n / ms / 1e6}
    opt = train.Adam(ds, {k: 1e-4 for k in train.PARAMS})
    elems = sum(getattr(ds, k).numel() for k in train.PARAMS)
    ms = _timed(lambda: opt.step(g, zero_grad=True), 20, 5, flush)
    out["adam_all_arrays_zero_grad"] = {"ms": ms, "bytes": 32 * elems, "GBps": 32 * elems / ms / 1e6, "launches": 6}
    cm = scenes.compact_model(N=n)
    dev = {k: (torch.from_numpy(v).cuda() if isinstance(v, np.ndarray) else v) for k, v in cm.items()}
    ms = _timed(lambda: train.decode_compact(dev, 3, 3, ds), 20, 5, flush)
    out["decode_compact"] = {"ms": ms, "bytes": (41 + 644) * n, "GBps": (41 + 644) * n / ms / 1e6,
                             "l2_gather_bytes": (8 * 564 + 6 * 12 + 3 * 6 * 16) * n}
    print(json.dumps(out), flush=True)


def sort_compare(flush):
    """north_star: "a hand-written device radix sort ... (CUB only as a comparison)".  For one view of cfg3 and of cfg4: the
    library's whole binning stage (compaction + tile grid + depth sort + offsets + pair emission + tile sort, CUDA events
    inside the library) next to cub::DeviceRadixSort::SortPairs over the same D pairs as literal 64-bit tile|depth keys
    (32 + ceil(log2 tiles) significant bits) — the single sort of [23]'s rasterizer, which additionally needs the key
    emission and a range-finding pass that are not timed here."""
    import ctypes as C
    import torch
    from paper_2412_20720_b200 import build, fdgs, scenes
    cmp_lib = C.CDLL(build.build_compare())
    cmp_lib.fdgs_cmp_cub_sort_pairs.argtypes = [C.c_void_p] * 4 + [C.c_int64, C.c_int, C.c_void_p, C.POINTER(C.c_size_t), C.c_void_p]
    for name, sc, cap in (("cfg3_video", scenes.multiview_video(n_views=1), 1 << 24), ("cfg4_driving", scenes.driving(n_views=1), 160 << 20)):
        ds = fdgs.DeviceScene.from_scene(sc)
        v = sc.views[0]
        r = fdgs.Renderer(ds, v.width, v.height, cap)
        cv = fdgs.make_view(v)
        fdgs.set_stage_timing(True)
        ours = {k: 0.0 for k in fdgs.STAGES[1:4]}
        reps = 1 if ONCE else 10
        for _ in range(reps + 2):
            flush.fill_(1)
            r.preprocess(cv)
            r.forward(cv)
            torch.cuda.synchronize()
            st = fdgs.stage_ms()
            if _ >= 2:
                for k in ours:
                    ours[k] += st[k] / reps
        fdgs.set_stage_timing(False)
        status = r.export(fdgs.EXPORT_STATUS)
        D = status["num_pairs"]
        keys_sorted = r.export(fdgs.EXPORT_SORTED_KEYS)[:D].contiguous()
        vals_sorted = r.export(fdgs.EXPORT_SORTED_VALS)[:D].contiguous()
        perm = torch.randperm(D, device="cuda")
        keys_in, vals_in = keys_sorted[perm].contiguous(), vals_sorted[perm].contiguous()
        keys_out, vals_out = torch.empty_like(keys_in), torch.empty_like(vals_in)
        tiles = ((v.width + 15) // 16) * ((v.height + 15) // 16)
        end_bit = 32 + max(1, (tiles - 1).bit_length())
        nbytes = C.c_size_t(0)
        stream = torch.cuda.current_stream().cuda_stream
        rc = cmp_lib.fdgs_cmp_cub_sort_pairs(None, None, None, None, D, end_bit, None, C.byref(nbytes), stream)
        assert rc == 0, rc
        temp = torch.empty(max(int(nbytes.value), 1), dtype=torch.uint8, device="cuda")

        def cub():
            rc = cmp_lib.fdgs_cmp_cub_sort_pairs(keys_in.data_ptr(), keys_out.data_ptr(), vals_in.data_ptr(), vals_out.data_ptr(), D,
                                                 end_bit, temp.data_ptr(), C.byref(nbytes), stream)
            assert rc == 0, rc
        ms_cub = _timed(cub, 10, 3, flush)
        torch.cuda.synchronize()
        same = bool(torch.equal(keys_out.view(torch.int64), keys_sorted.view(torch.int64)))
        print(json.dumps({"config": "sort_compare_" + name, "N": sc.N, "pairs": D, "visible": status["num_visible"], "key_bits": end_bit,
                          "ours_ms": ours, "ours_total_ms": sum(ours.values()),
                          "ours_sorts_only_ms": ours["sort_depth"] + ours["tile_lists"],
                          "cub_sortpairs_64bit_ms": ms_cub, "cub_keys_equal_ours": same,
                          "note": "ours_total includes compaction, tile ranges, offsets and pair emission; the CUB figure is the sort alone"}),
              flush=True)
        del r, ds, keys_in, vals_in, keys_out, vals_out, keys_sorted, vals_sorted, perm, temp
        torch.cuda.empty_cache()


def full_training_step(flush):
    """cfg3 step with the optimiser inside the timed region: fdgs_step_batch (4 views) + fdgs_regularizers + dense Adam over
    all six arrays (gradients cleared by the Adam pass)."""
    import torch
    from paper_2412_20720_b200 import fdgs, scenes, train
    sc = scenes.multiview_video()
    ds = fdgs.DeviceScene.from_scene(sc)
    v0 = sc.views[0]
    bs = fdgs.BatchStep(ds, v0.width, v0.height, 1 << 24, len(sc.views))
    cvs = [fdgs.make_view(v) for v in sc.views]
    for i, rr in enumerate(bs.renderers):
        rr.target_dev.copy_(torch.from_numpy(scenes.target_image(sc.seed, i, v0.width, v0.height)).cuda())
    g = ds.zero_grads()
    opt = train.Adam(ds, {k: 1e-6 for k in train.PARAMS})

    def render_only():
        for a in g.values():
            if a is not None:
                a.zero_()
        bs.step(cvs, g)

    def step():
        bs.step(cvs, g)
        train.regularizers(ds, g, lambda_sparse=1e-4, lambda_covt=1e-4)
        opt.step(g, zero_grad=True)
    ms0 = _timed(render_only, 10, 3, flush)
    ms1 = _timed(step, 10, 3, flush)
    print(json.dumps({"config": "cfg3_full_training_step", "N": sc.N, "views_per_step": len(sc.views),
                      "render_fwd_bwd_ms": ms0, "with_regularizers_and_adam_ms": ms1, "steps_per_s_with_optimizer": 1e3 / ms1}), flush=True)


def feature_terms(flush, n=1_000_000, C=32):
    """Feature channels (D = 32) and optical flow at cfg3's size, view 0: ms per call next to the colour
    forward / backward of the same view."""
    import torch
    from paper_2412_20720_b200 import fdgs, scenes
    sc = scenes.multiview_video(N=n, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    v = sc.views[0]
    r = fdgs.Renderer(ds, v.width, v.height, 1 << 24)
    cv = fdgs.make_view(v)
    r.preprocess(cv, sync=True)
    r.forward(cv)
    feat = torch.randn((n, C), device="cuda")
    G = torch.randn((C, v.height, v.width), device="cuda")
    gf, g = torch.zeros_like(feat), ds.zero_grads()
    out = {"config": "feature_terms", "N": n, "C": C, "width": v.width, "height": v.height}
    out["colour_forward_ms"] = _timed(lambda: r.forward(cv), 10, 3, flush)
    out["colour_backward_ms"] = _timed(lambda: r.backward(cv, G[:3].contiguous(), g), 10, 3, flush)
    out["features_forward_ms"] = _timed(lambda: r.features_forward(cv, feat), 10, 3, flush)
    out["features_backward_ms"] = _timed(lambda: r.features_backward(cv, feat, G, gf, g), 10, 3, flush)
    out["features_backward_feat_only_ms"] = _timed(lambda: r.features_backward(cv, feat, G, gf, None), 10, 3, flush)
    out["splat_flow_ms"] = _timed(lambda: r.splat_flow(cv, 1.0 / 30.0), 10, 3, flush)
    flow = r.splat_flow(cv, 1.0 / 30.0)
    out["flow_map_forward_ms"] = _timed(lambda: r.features_forward(cv, flow), 10, 3, flush)
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--frames", type=int, default=24)
    ap.add_argument("--max-n", type=int, default=8_000_000)
    ap.add_argument("--skip-train", action="store_true")
    ap.add_argument("--skip-sweep", action="store_true")
    ap.add_argument("--once", action="store_true", help="one warm-up and one timed iteration per operation (for ncu captures)")
    ap.add_argument("--sort-compare", action="store_true", help="binning stage vs cub::DeviceRadixSort on 64-bit keys (comparison only)")
    ap.add_argument("--train-terms", action="store_true", help="time the f2-f4 kernels (mask, regularisers, Adam, decode) only")
    args = ap.parse_args()
    global ONCE
    ONCE = args.once
    import torch
    from paper_2412_20720_b200 import build, scenes
    if not torch.cuda.is_available():
        raise RuntimeError("sweep needs a CUDA device: the product has no CPU fallback")
    build.build()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    if args.sort_compare:
        sort_compare(flush)
        return
    if args.train_terms:
        train_terms(flush)
        feature_terms(flush)
        full_training_step(flush)
        return
    if not args.skip_train:
        train_cfg("cfg2_object", scenes.single_object(), 1 << 22, flush)
        train_cfg("cfg4_driving", scenes.driving(), 160 * 1024 * 1024, flush)
    if not args.skip_sweep:
        sweep_cfg5(args.frames, args.max_n, flush)


if __name__ == "__main__":
    main()
