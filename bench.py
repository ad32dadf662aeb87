#!/usr/bin/env python
"""bench.py — BASELINE.json's metric on its headline config: forward+backward steps/s (and forward FPS) of the
time-sliced tile rasterizer at 1M 4D Gaussians, 1352x1014, batch of 4 views (cfg3), seeded synthetic data.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

One JSON line on stdout (rank 0).  `value` = steps/s with everything resident in HBM; `e2e` = the same through
fdgs_step_batch with pinned HOST target images copied in and the per-view losses read back every step; `roofline` = the dominant kernel
against the ALU issue roof derived in DESIGN.md (both per-unit instruction models printed); `cpu_baseline` = the float64
oracle on this box's host cores: one full step on all cores plus one view single-threaded, per stage.  --impl reference
times that oracle as the reference arm, one full step (all four views) per timed step.
Multi-GPU: the path does not shard: N ranks render N independent replicas.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fwd+bwd steps/s, 1M 4D Gaussians @1352x1014, batch of 4 views"
WORKLOAD = "cfg3_video: N=1M, K=48 (L=3 x n_time=3), 1352x1014, fov 60, 4 jittered views at 4 seeded times, L1 loss"
PAIR_CAPACITY = 16 * 1024 * 1024
SM_COUNT, LANES_PER_SM, SM_MAX_HZ = 148, 128, 1.965e9
ALU_PEAK_TLANE = SM_COUNT * LANES_PER_SM * SM_MAX_HZ / 1e12      # 37.2 T lane-instructions/s
# DRAM bytes per launch of the dominant kernel: NOT measured by this run (ncu counters cannot be read from inside it).
# The value is read from the committed ncu --set full summary named here and is labelled as such in the JSON line.
TRAFFIC_SOURCE = os.path.join(ROOT, "profiles", "r2_blend_traffic.json")


def ncu_traffic(kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed capture, with its provenance."""
    try:
        with open(TRAFFIC_SOURCE) as f:
            d = json.load(f)
        return float(d["kernels"][kernel]["dram_bytes_per_launch"]), "ncu --set full capture, " + d["source"]
    except Exception:
        return None, "no committed ncu capture for this kernel"


def bench_config(stress=False):
    """The `config` object of the JSON line: identical for the product arm and for the reference (oracle) arm, which runs
    the same workload (the keys about the GPU schedule simply do not apply to it)."""
    return {"workload": WORKLOAD, "stress_variant": bool(stress), "pair_capacity": PAIR_CAPACITY,
            "l2": "256 MB flush write between timed steps; parameters (644 MB) exceed L2", "multi_gpu": "replicas only",
            "schedule": "fdgs_step_batch: the 4 views on 4 worker streams and workspaces; backward preprocess of the batch after the last blend (one colour pass over the union of the views' survivors, geometry view after view)"}


def hbm_peak():
    """Measured copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def stage_rooflines(stage, work, N, K, n_views):
    """Every stage against its own roof: algorithmic bytes / CUDA-event time vs the HBM copy peak for
    the memory-bound stages, algorithmic lane-instructions vs the ALU issue peak for the two blend kernels."""
    peak, src = hbm_peak()
    nv, D = work["visible"], work["pairs"]          # summed over the views of the step
    # the public fdgs_preprocess / fdgs_render_forward pair (timed here stage by stage) evaluates the colour of a degree-3
    # scene in a kernel of its own on a side stream, under the depth sort and the row scatter: two rows
    byts = {"preprocess": n_views * 72 * N + nv * 76,               # geometry rows of every primitive; record, hand-over, rectangle of the survivors
            "colour_side_stream": nv * (12 * K + 4 + 16 + 12),      # coefficient rows of the survivors; id and hand-over read, three colour slots written
            "compact+tile_grid": n_views * 4 * N + 16 * nv,
            "sort_depth": 4 * 16 * nv,
            "tile_lists": 12 * nv + 4 * D,                    # ids and rectangles of the survivors read, 4 B written per pair
            "preprocess_bwd": nv * (36 + 68 + 12 * K + 2 * (12 * K + 68) + 64)}
    out = {}
    for k, b in byts.items():
        if not stage.get(k, 0.0) > 0.0:
            continue
        gbs = b / (stage[k] * 1e-3) / 1e9
        out[k] = {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "frac_of_8tbs_spec": gbs / 8000.0,
                  "algorithmic_bytes": b}
    out["peak_source_hbm"] = src
    return out




class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200"], stdout=subprocess.PIPE, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=2)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        reasons = set()
        for r in self.rows:
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if val == "Active":
                    reasons.add(name)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(self.rows[0][1]) if self.rows and self.rows[0][1].isdigit() else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(local_ms: float, world: int, device="cpu") -> float:
    """The step time of a multi-rank run is the slowest rank's (all-reduce MAX over the process group)."""
    if world <= 1:
        return float(local_ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def whole_job_value(world: int, ms_per_step: float) -> float:
    """Replicas only: every rank renders its own full step, so the job does `world` steps per step time."""
    return world * 1e3 / ms_per_step


ORACLE_STAGES = ("preprocess+lists", "blend_fwd", "loss+backward")


def oracle_step_seconds(scene, view_indices, threads=None):
    """The oracle as it stands: preprocess (A1-A8) + forward blend + L1 gradient + backward of the given views on the host
    cores.  Returns (seconds per stage summed over the views, threads used)."""
    import numpy as np
    import oracle
    from paper_2412_20720_b200 import scenes
    if threads:
        oracle.set_num_threads(threads)
    o = oracle.Oracle(**scene.arrays(), sh_degree=scene.sh_degree, n_time=scene.n_time)
    per = dict.fromkeys(ORACLE_STAGES, 0.0)
    for vi in view_indices:
        v = scene.views[vi]
        tgt = scenes.target_image(scene.seed, vi, v.width, v.height).astype(np.float64)
        t0 = time.perf_counter()
        o.preprocess(v.view, (v.fx, v.fy, v.cx, v.cy), v.width, v.height, v.t, v.period_T, v.bg)
        t1 = time.perf_counter()
        img = o.forward()[0]
        t2 = time.perf_counter()
        o.backward(np.sign(img - tgt) / img.size)
        t3 = time.perf_counter()
        per["preprocess+lists"] += t1 - t0; per["blend_fwd"] += t2 - t1; per["loss+backward"] += t3 - t2
    return per, oracle.num_threads()


def run_reference(args):
    """Reference arm = the float64 oracle (there is no upstream code).  Rank 0 only.  Every warm-up and timed step is one
    REAL step: all views of the batch, nothing extrapolated (about 10 s per step on 16 cores)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2412_20720_b200 import scenes
    scene = scenes.multiview_video(quat_mode="random") if args.stress else scenes.multiview_video()
    n_views = len(scene.views)
    secs, cores, stages = [], 0, dict.fromkeys(ORACLE_STAGES, 0.0)
    for it in range(args.warmup + args.steps):
        per, cores = oracle_step_seconds(scene, range(n_views))
        if it >= args.warmup:
            secs.append(sum(per.values()))
            for k in stages:
                stages[k] += per[k] / args.steps
    ms_step = 1e3 * sum(secs) / len(secs)
    val = 1e3 / ms_step
    sample = f"every step = all {n_views} views of cfg3 (preprocess+forward+L1+backward at N=1M, 1352x1014), no extrapolation"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": "steps/s", "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f64", "data": "synthetic", "config": bench_config(args.stress),
                      "cpu_baseline": {"value": val, "unit": "steps/s", "cores": cores, "kind": "oracle", "sample": sample,
                                       "stage_seconds_per_step": stages},
                      "e2e": {"value": val, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def run_fdgs(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2412_20720_b200 import build, fdgs, scenes
    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    build.build()
    # --stress: SURVEY 8(d) "run cfg3 additionally with cfg1-style fully random q_r as a stress variant and report both"
    scene = scenes.multiview_video(quat_mode="random") if args.stress else scenes.multiview_video()
    views = scene.views
    n_views = len(views)
    ds = fdgs.DeviceScene.from_scene(scene, device=dev)
    bs = fdgs.BatchStep(ds, views[0].width, views[0].height, PAIR_CAPACITY, n_views)     # one workspace per view of the batch
    r = bs.renderers[0]
    cviews = [fdgs.make_view(v) for v in views]
    tg_np = [scenes.target_image(scene.seed, i, views[0].width, views[0].height) for i in range(n_views)]
    targets = [torch.from_numpy(t).to(dev) for t in tg_np]
    targets_host = [torch.from_numpy(t).pin_memory() for t in tg_np]
    loss_host = torch.zeros(n_views).pin_memory()
    for rr, tg in zip(bs.renderers, targets):
        rr.target_dev.copy_(tg)
    grads = ds.zero_grads()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def zero_grads():
        for g in grads.values():
            if g is not None:
                g.zero_()

    def step_device():       # fdgs_step_batch, targets resident in HBM, nothing read back; gradients zeroed inside the call
        bs.step(cviews, grads, zero_grads=True)

    def step_host():         # fdgs_step_batch with pinned HOST targets copied in and the four losses copied back (synchronises)
        bs.step(cviews, grads, targets_host=targets_host, loss_host=loss_host, zero_grads=True)

    def forward_only(cv):
        r.preprocess(cv)
        r.forward(cv)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, steps, warmup):
        """per-step CUDA events on the launching stream; L2 flushed (outside the events) between steps"""
        for _ in range(warmup):
            fn()
        barrier()
        evs = []
        for _ in range(steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            evs.append((e0, e1))
        barrier()
        ms = [a.elapsed_time(b) for a, b in evs]
        return max_over_ranks(sum(ms), world, dev) / steps, ms

    # ---- headline: fwd+bwd steps/s, inputs resident in HBM -------------------------------------------------
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)
    l0 = fdgs.launch_count()
    ms_step, _ = timed(step_device, args.steps, args.warmup)
    launches = (fdgs.launch_count() - l0) * args.steps // (args.steps + args.warmup)
    # the driver fixes K (20 steps = 0.1 s): a second, sustained region of 1 s next to it, same clock sampler
    sustained_steps = max(args.steps, 200)
    ms_sustained, _ = timed(step_device, sustained_steps, 0)
    clocks = sampler.stop() if sampler else None
    for rr in bs.renderers:
        status = rr.export(fdgs.EXPORT_STATUS)
        if status["overflow"]:
            raise RuntimeError(f"pair capacity {PAIR_CAPACITY} exceeded: {status}")
    loss_dev = float(bs.loss.sum())
    # ---- end to end through the C ABI with host buffers ----------------------------------------------------
    ms_e2e, _ = timed(step_host, max(3, args.steps // 2), 3)
    # ---- forward-only FPS (one frame = preprocess + forward of one view) -----------------------------------
    fps_ms, fps_all = [], []
    for cv in cviews:
        m, per = timed(lambda: forward_only(cv), 25, 20)      # 20 warm-up + 25 timed frames per view: 100 timed frames
        fps_ms.append(m)
        fps_all += per
    ms_frame = sum(fps_ms) / len(fps_ms)
    fps_all.sort()
    # ---- playback throughput: consecutive frames in flight on separate streams / workspaces (cfg5-style free-viewpoint
    # video): the scans and sorts of frame k+1 overlap the blend of frame k -------------------------------
    streams = [torch.cuda.Stream() for _ in range(n_views)]
    n_frames = 40

    def playback():
        main = torch.cuda.current_stream()
        ev = torch.cuda.Event()
        ev.record(main)
        for k in range(n_frames):
            s_, rr = streams[k % n_views], bs.renderers[k % n_views]
            s_.wait_event(ev)
            with torch.cuda.stream(s_):
                rr.preprocess(cviews[k % n_views])
                rr.forward(cviews[k % n_views])
        for s_ in streams:
            e = torch.cuda.Event()
            e.record(s_)
            main.wait_event(e)

    ms_playback, _ = timed(playback, 5, 3)
    ms_frame_pipelined = ms_playback / n_frames
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- per-stage times (events at the stage boundaries inside the library), one view at a time -----------
    # one untimed pass first: the view-by-view backward launches kernels that fdgs_step_batch never used (their first launch
    # loads the module: milliseconds, which would land in one repetition of one stage)
    r.preprocess(cviews[0]); r.forward(cviews[0]); r.l1_loss(targets[0]); r.backward(cviews[0], r.dL_dimage, grads)
    torch.cuda.synchronize()
    fdgs.set_stage_timing(True)
    stage = {k: 0.0 for k in fdgs.STAGES}
    work = {"walk": 0, "exp": 0, "comp": 0, "staged": 0, "walk_bwd": 0, "pairs": 0, "visible": 0}
    reps = 5
    for cv, tg in zip(cviews, targets):
        for _ in range(reps):
            flush.fill_(1)
            r.preprocess(cv); r.forward(cv); r.l1_loss(tg); r.backward(cv, r.dL_dimage, grads)
            for k, v in fdgs.stage_ms().items():
                stage[k] += v / reps
        w = r.blend_stats(cv)
        st = r.export(fdgs.EXPORT_STATUS)
        work["walk"] += w[0]; work["exp"] += w[1]; work["comp"] += w[2]; work["staged"] += w[3]
        work["walk_bwd"] += int(r.n_contrib.sum()); work["pairs"] += st["num_pairs"]; work["visible"] += st["num_visible"]
    fdgs.set_stage_timing(False)
    # ---- roofline of the dominant kernel (algorithmic lane-instructions / measured time) ----
    # Two per-unit models on the SAME measured work counters (pairs walked / reaching exp2 / composited):
    #   "builder": forward 8 per walked pair + 3 per exp2 + 7 per composite; backward 8 + 3 + 50
    #   "survey":  forward 13 per walked pair (12-14 incl. the MUFU) + 8 per composite; backward 14 per walked + (50 + 2 MUFU - 14) more
    #              per composite
    # `frac` (the headline) uses the builder's model, which is the stricter of the two.
    frac_exp = work["exp"] / max(work["walk"], 1)
    models = {"builder": {"fwd": 8 * work["walk"] + 3 * work["exp"] + 7 * work["comp"],
                          "bwd": 8 * work["walk_bwd"] + 3 * frac_exp * work["walk_bwd"] + 50 * work["comp"]},
              "survey": {"fwd": 13 * work["walk"] + 8 * work["comp"],
                         "bwd": 14 * work["walk_bwd"] + (52 - 14) * work["comp"]}}
    instr_fwd, instr_bwd = models["builder"]["fwd"], models["builder"]["bwd"]
    dom = "blend_bwd" if stage["blend_bwd"] >= stage["blend_fwd"] else "blend_fwd"
    key = "bwd" if dom == "blend_bwd" else "fwd"
    kernel = "blend_bwd2_kernel" if dom == "blend_bwd" else "blend_fwd_kernel"
    instr = models["builder"][key]
    achieved = instr / n_views / (stage[dom] / n_views * 1e-3) / 1e12
    traffic, traffic_src = ncu_traffic(kernel)
    peaks = fdgs.measure_peaks()           # measured FMA / MUFU pipe peaks next to the derived ALU roof
    roofline = {"kernel": kernel, "bound": "alu", "achieved": achieved,
                "peak": ALU_PEAK_TLANE, "unit": "Tlane-instr/s", "frac": achieved / ALU_PEAK_TLANE,
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "DERIVED, not measured: 148 SMs x 128 FP32 lanes x 1.965 GHz (B200_PROFILING.md unit counts and max clock)",
                "peak_measured_fma_tlane_per_s": peaks["fma_tlane_per_s"], "peak_measured_mufu_ex2_t_per_s": peaks["mufu_ex2_t_per_s"],
                "frac_of_measured_fma_peak": achieved / max(peaks["fma_tlane_per_s"], 1e-9),
                "model": "builder (8/+3/+7 forward, 8/+3/+50 backward lane-instr per walked / exp2 / composited pair)",
                "frac_by_model": {m: models[m][key] / (stage[dom] * 1e-3) / 1e12 / ALU_PEAK_TLANE for m in models},
                "counters_per_step": {"walked_fwd": work["walk"], "exp2": work["exp"], "composited": work["comp"], "walked_bwd": work["walk_bwd"]},
                "algorithmic_lane_instr_per_launch": instr / n_views, "ms_per_launch": stage[dom] / n_views}
    per_stage = stage_rooflines(stage, work, ds.N, ds.K, n_views)
    for name, k2 in (("blend_fwd", "fwd"), ("blend_bwd", "bwd")):
        a = models["builder"][k2] / (stage[name] * 1e-3) / 1e12
        per_stage[name] = {"bound": "alu", "achieved": a, "peak": ALU_PEAK_TLANE, "unit": "Tlane-instr/s", "frac": a / ALU_PEAK_TLANE,
                           "frac_survey_model": models["survey"][k2] / (stage[name] * 1e-3) / 1e12 / ALU_PEAK_TLANE,
                           "algorithmic_lane_instr": models["builder"][k2]}
    # ---- CPU baseline: the oracle, one full step on all cores + one view on a single thread, per stage ----------
    cpu = None
    if not args.no_cpu_baseline:
        per_all, cores = oracle_step_seconds(scene, range(n_views))
        tot = sum(per_all.values())
        per_one, _ = oracle_step_seconds(scene, [0], threads=1)
        import oracle as _o
        _o.set_num_threads(cores)
        cpu = {"value": 1.0 / tot, "unit": "steps/s", "cores": cores, "kind": "oracle",
               "sample": f"one full step: all {n_views} views (preprocess+forward+L1+backward at N=1M, 1352x1014) in {tot:.1f} s on {cores} threads; "
                         f"single-thread figures: view 0 only ({sum(per_one.values()):.1f} s)",
               "stage_seconds_per_step_all_cores": per_all,
               "single_thread": {"cores": 1, "sample": "view 0 of the step (1 of 4 views)", "stage_seconds_per_view": per_one,
                                 "steps_per_s_extrapolated_x4": 1.0 / (n_views * sum(per_one.values()))}}
    img_bytes = 3 * views[0].width * views[0].height * 4
    out = {"metric": METRIC, "value": whole_job_value(world, ms_step), "unit": "steps/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": bench_config(args.stress),
           "replicas": {"n": world, "value_per_replica": 1e3 / ms_step,
                        "note": "replicas only (DESIGN.md section 7): `value` is N independent copies of the single-GPU step, not one sharded job"},
           "sustained": {"steps": sustained_steps, "ms_per_step": ms_sustained, "value": whole_job_value(world, ms_sustained)},
           "forward_fps": world * 1e3 / ms_frame, "ms_per_frame": ms_frame,
           "ms_per_frame_median": fps_all[len(fps_all) // 2], "ms_per_frame_min": fps_all[0], "frames_timed": len(fps_all),
           "forward_fps_pipelined": world * 1e3 / ms_frame_pipelined, "ms_per_frame_pipelined": ms_frame_pipelined,
           "e2e": {"value": world * 1e3 / ms_e2e, "unit": "steps/s", "h2d_bytes_per_step": n_views * img_bytes, "d2h_bytes_per_step": n_views * 4,
                   "ms_per_step": ms_e2e},
           "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
           "stage_ms_per_step": stage, "stage_rooflines": per_stage, "work_per_step": work, "loss": loss_dev,
           "paper_context": "114 FPS forward on Plenoptic Video, hardware not named (PAPER.md Table 1, L347) - context only"}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="fdgs", choices=["fdgs", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--stress", action="store_true", help="cfg3 with fully random q_r (SURVEY 8(d) stress variant)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "fdgs" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_fdgs(args)


if __name__ == "__main__":
    main()
