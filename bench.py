#!/usr/bin/env python
"""bench.py -- secondary-ray MRay/s of the hot path on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload interior|landscape|cornell] [--impl reference]

A step = one frame of the whole hot path: crt_trace_primary -> crt_shade_accumulate(0) ->
for b = 1..B { crt_generate_secondary(b) -> crt_trace -> crt_shade_accumulate(b) } on one batch of synthetic input
(default workload: BASELINE config 2, the interior scene at 1920x1080, 1 spp, 2 bounces, groups 4x4, stride 4, seed 1).
`value` = live secondary rays of the K timed steps / their device time, for mode direct_reuse, with `--frames-in-flight` (default 3)
frames rendered concurrently, each on its own context and stream (config.single_stream_value = one frame at a time); the other modes
and the stage-level numbers (generate / encode+sort+permute / trace), all one frame at a time, are in "modes".  See DESIGN.md section 7.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "secondary_ray_throughput"
UNIT = "MRay/s"
WORKLOADS = {
    # name: (scene kwargs, w, h, spp, bounces, gw, gh, stride, seed, BASELINE config index)
    "cornell": ("cornell", dict(seed=0), 64, 64, 1, 1, 4, 4, 2, 0, 0),
    "interior": ("interior", dict(seed=1), 1920, 1080, 1, 2, 4, 4, 4, 1, 1),
    "landscape": ("landscape", dict(seed=2), 1920, 1080, 1, 2, 4, 4, 4, 2, 3),
}
# FLOPs of the traversal kernel per unit of work, counted from csrc/trace.cu: a node visit tests two
# child boxes = 12 (subtract, multiply) pairs + 2 inflations = 26 flop (min/max/compare are not flops); a triangle test
# (Moller-Trumbore as written in crt_device.cuh) = 2 cross (9 each) + 4 dot (5 each) + 1 subtract-vector (3) + 1 reciprocal (1)
# + 3 scalings (3) + 1 add (1) = 46 flop.  Ray setup of the 16-bit-node kernel: 3 reciprocals, 3 scalings of them, origin into grid
# units (3 subtract + 3 multiply), 3 x (multiply + FMA) for the plane constants = 21 flop per ray.  (A node visit of the 16-bit
# layout is the same 12 FMA + the prune-bound multiply; the PRMT plane decode is not a flop.)
FLOP_PER_NODE_VISIT, FLOP_PER_TRI_TEST, FLOP_PER_RAY = 26.0, 46.0, 21.0
# nominal FP32 peak from the guide's unit counts: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz (B200_PROFILING.md table)
FP32_PEAK_TFLOPS_NOMINAL = 148 * 128 * 2 * 1.965e9 / 1e12
# ncu-measured figures of the dominant kernel (trace_dyn_kernel<0,1>, secondary rays in direct_reuse order), per LIVE ray, mean of the bounce-1 and
# bounce-2 launches of one frame; carried over from the named profile (ncu replays kernels, so these cannot be taken inside a timed run):
#   flop  = smsp__sass_thread_inst_executed_op_fadd_pred_on.sum + ..fmul.. + 2 x ..ffma...  ncu does not count the packed FFMA2 the default
#           kernel now uses under op_ffma, so the counters are taken on the scalar-FFMA instantiation (trace_kernel 4: the same 12 fused multiply-adds per
#           node visit and the same triangle test; its ray setup has 12 more)
#   dram  = dram__bytes_read.sum + dram__bytes_write.sum of the default kernel
NCU_PER_RAY = {
    "interior": {"flop": 1673.0, "dram_bytes": 62.0, "source": "profiles/r02o_device_reinsertion.md (ncu on the default tree: host SAH, large triangles pre-split, parallel re-insertion on the device at single-reference granularity; flop: 6.512 G over 3,891,381 live rays of frame 7; dram: 241.3 MB over the same rays; the plain SAH tree: 1,897 flop per ray, profiles/r02c)"},
    "landscape": {"flop": 1370.0, "dram_bytes": 102.9, "source": "profiles/r02o_device_reinsertion.md (same commit; flop: 2.792 G over 2,037,200 live rays of frame 7; dram: 209.6 MB over the same rays; the plain SAH tree: 1,383, profiles/r02c)"},
}
# what ncu shows to be the kernel's limiter (not modelled by the two-term roofline): profiles/r02a, r02c
TRACE_LIMITER = {
    "interior": {"unit": "half-rate ALU pipe (plane decode, min/max, selects: 32 of 52 instructions per node visit) under long-scoreboard stalls of divergent 256-bit node gathers at 32 resident warps per SM", "top_stall": "long_scoreboard: 5.4-6.7 warps per issued instruction",
                 "issue_slots_busy_pct": 61.2, "active_threads_per_warp_instruction": 16.1, "l1_sector_hit_pct": 66.4, "l2_sector_hit_pct": 75.1, "alu_pipe_pct": 53.4, "fma_pipe_pct": 23.5,
                 "l1tex__data_pipe_lsu_wavefronts_pct_of_peak": 56.4, "dram_pct": 2.0, "source": "profiles/r02c_roofline_inputs.md (mean of the bounce-1 and bounce-2 launches); profiles/r02a for the experiments behind the reading"},
    "landscape": {"unit": "as interior; bounce 2 (0.42 M live rays of 2.09 M slots) is a short launch dominated by its tail", "top_stall": "long_scoreboard: 5.2 (bounce 1) / 10.1 (bounce 2) warps per issued instruction",
                  "issue_slots_busy_pct": 51.4, "active_threads_per_warp_instruction": 15.7, "l1_sector_hit_pct": 58.9, "l2_sector_hit_pct": 59.7, "alu_pipe_pct": 47.3, "fma_pipe_pct": 17.9,
                  "l1tex__data_pipe_lsu_wavefronts_pct_of_peak": 41.9, "dram_pct": 3.9, "source": "profiles/r02c_roofline_inputs.md (mean of the two launches)"},
}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


def _scene(workload, scale=1):
    import crt_inputs as I
    name, kw, w, h, spp, nb, gw, gh, s, seed, cfg = WORKLOADS[workload]
    scene = I.by_name(name, **kw)
    w, h = max(w // scale, 8), max(h // scale, 8)
    return scene.with_camera(w, h), (w, h, spp, nb, gw, gh, s, seed, cfg)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in self.rows if len(r) >= 7 for k in range(4) if r[3 + k].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons, "samples": len(sm)}


_SWEEP_CLOCKS = None      # clock sampler of a --sweep run (started in main(), stopped where the sweep prints its JSON line)


# ------------------------------------------------------------------------------------------------ reference arm (oracle)
def run_reference(args):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the same workload: the same scene and
    camera at 1/4 x 1/4 of the resolution (1/16 of the pixels), same spp / bounces / grouping, one frame per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as O
    O.build()
    scale = 4
    scene, (w, h, spp, nb, gw, gh, s, seed, cfg) = _scene(args.workload, scale)
    bvh = O.Bvh(scene.verts)
    steps, warm = max(1, min(args.steps, 3)), min(args.warmup, 1)
    rays = 0; secs = 0.0
    for i in range(warm + steps):
        t0 = time.perf_counter()
        _, times, counts = O.render_frame(bvh, scene, O.frame(w, h, spp, seed, i), nb, 2, gw, gh, s)
        dt = time.perf_counter() - t0
        if i >= warm:
            rays += int(counts[0]); secs += dt
    v = rays / secs / 1e6
    sample = f"{steps} frame(s) of the {args.workload} scene at {w}x{h} (1/{scale * scale} of the pixels), {spp} spp, {nb} bounces, direct_reuse {gw}x{gh} stride {s}"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps, "warmup": warm,
            "ms_per_step": 1e3 * secs / steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"BASELINE config {cfg + 1}: {args.workload} (bounded sample)", "sample": sample, "mode": "direct_reuse"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def cpu_baseline(workload):
    import oracle as O
    O.build()
    scale = 1 if workload != "landscape" else 2       # the full 1920x1080 frame; the landscape's 10.3 M-triangle tree takes the single-threaded builder minutes: 1/4 of the pixels there
    scene, (w, h, spp, nb, gw, gh, s, seed, cfg) = _scene(workload, scale)
    bvh = O.Bvh(scene.verts)
    t0 = time.perf_counter()
    _, times, counts = O.render_frame(bvh, scene, O.frame(w, h, spp, seed, 0), nb, 2, gw, gh, s)
    dt = time.perf_counter() - t0
    return {"value": counts[0] / dt / 1e6, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"1 frame of the {workload} scene at {w}x{h} ({'the full frame' if scale == 1 else '1/%d of the pixels' % (scale * scale)}), {spp} spp, {nb} bounces, direct_reuse {gw}x{gh} stride {s}; "
                      f"{int(counts[0])} secondary rays in {dt:.2f} s (trace {times[1]:.2f} s, generate {times[0]:.2f} s); BVH build untimed",
            "secondary_trace_only_mray_s": counts[0] / max(times[1], 1e-9) / 1e6,
            "node_visits_per_ray": counts[1] / max(counts[0], 1), "tri_tests_per_ray": counts[2] / max(counts[0], 1)}


# ------------------------------------------------------------------------------------------------ CUDA arm
def reduce_over_ranks(ms, rays, device, world):
    """Whole-job figures of N independent replicas: time = MAX over ranks, rays = SUM over ranks.
    The only collectives of the bench; there is none on the data path."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device); r = torch.tensor([rays], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX); dist.all_reduce(r, op=dist.ReduceOp.SUM)
    return float(t.item()), float(r.item())


def replica_frame_index(step, rank, world):
    """Replicas render disjoint frame indices so that no two ranks repeat the same work."""
    return step * world + rank


def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_2310_07182_b200 as crt

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    ctx = crt.Context(local)
    options = [o.split("=") for o in args.set]
    for k_, v_ in options:
        ctx.crt_set_option(k_, int(v_))
    scene, (w, h, spp, nb, gw, gh, s, seed, cfg) = _scene(args.workload)
    t0 = time.perf_counter()
    bvh = ctx.crt_build_bvh(scene.verts, scene.mat_id, **BVH_KW)
    build_s = time.perf_counter() - t0
    info = bvh.info()
    mats_dev = ctx.upload(scene.materials)
    mats = ctx.scene_mats(mats_dev, len(scene.materials), scene.env)
    cam = crt.make_camera(scene.camera)
    stream = torch.cuda.current_stream()
    K, W = args.steps, args.warmup

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def time_mode(mode, host=False, stages=True):
        """W warm-up + K timed frames of one mode; replicas (rank r) render different frame indices.  stages=False: no per-stage events (the
        library then runs a frame in bands, option frame_bands)."""
        order = crt.make_order(mode, gw, gh, s)
        n_paths, n_slots, _ = crt.crt_layout(crt.make_frame(w, h, spp), order)
        ws = ctx.frame_workspace(crt.make_frame(w, h, spp), order, host_materials=len(scene.materials) if host else 0)
        nsec = torch.zeros((K + W, max(nb, 1)), dtype=torch.int32, device=ctx.device)
        stage = np.zeros(8, np.float32); bounce_ms = np.zeros((max(nb, 1), 3), np.float32)
        if host:
            accum_h = torch.zeros((h, w, 3), dtype=torch.float32).pin_memory()
            nsec_h = np.zeros((K + W, max(nb, 1)), np.uint32)
            mats_h = scene.materials
        else:
            accum = torch.zeros((h, w, 3), device=ctx.device)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def step(i, rec):
            fr = crt.make_frame(w, h, spp, seed, replica_frame_index(i, rank, world))
            if host:
                ctx.crt_render_frame_host_resident(bvh, mats_h, scene.env, cam, fr, order, nb, i == 0, accum_h, nsec_h[i], ws)
            else:
                ctx.crt_render_frame(bvh, mats, cam, fr, order, nb, accum, ws, n_secondary=nsec[i], record_times=rec)
                if rec:
                    ctx.crt_frame_times(stage)        # synchronises the frame's last event; the K steps still run back to back on the device
                    ctx.crt_frame_bounce_times(nb, bounce_ms)
        for i in range(W):
            step(i, False)
        barrier()
        e0.record(stream)
        for i in range(W, W + K):
            step(i, stages and not host)
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        rays = int(nsec_h[W:].sum()) if host else int(nsec[W:].sum().item())
        ms_all, rays_all = reduce_over_ranks(ms, rays, ctx.device, world)
        res = {"mray_s": rays_all / (ms_all * 1e-3) / 1e6, "ms_per_step": ms_all / K, "secondary_rays_per_step": rays / K, "n_slots": n_slots}
        if not host and stages:
            sec_ms = float(stage[2] + stage[3])       # generate(+encode+sort+permute) + secondary trace, summed over the K steps (this rank)
            res.update({"secondary_loop_mray_s": rays / (sec_ms * 1e-3) / 1e6, "trace_only_mray_s": rays / (float(stage[3]) * 1e-3) / 1e6,
                        "primary_ms": float(stage[0]) / K, "shade_ms": float(stage[1]) / K, "generate_ms": float(stage[2] - stage[4]) / K,
                        "encode_sort_permute_ms": float(stage[4]) / K, "trace_ms": float(stage[3]) / K, "trace_launch_ms": float(stage[3]) / (K * max(nb, 1))})
            nsb = nsec[W:].sum(0).cpu().numpy().astype(np.float64)          # live rays per bounce over the K steps
            res["per_bounce"] = [{"bounce": b + 1, "rays_per_step": float(nsb[b]) / K, "generate_ms": float(bounce_ms[b, 0]) / K, "encode_sort_permute_ms": float(bounce_ms[b, 1]) / K,
                                  "trace_ms": float(bounce_ms[b, 2]) / K, "trace_only_mray_s": float(nsb[b]) / max(float(bounce_ms[b, 2]) * 1e-3, 1e-12) / 1e6,
                                  "loop_mray_s": float(nsb[b]) / max(float(bounce_ms[b].sum()) * 1e-3, 1e-12) / 1e6} for b in range(nb)]
        return res

    # ---- frames in flight: F contexts (one per stream; a crt_ctx serialises its own calls) render alternate frames concurrently, so the
    # tail of one traversal launch (stragglers after the ray queue is empty: about 0.1 ms per launch, profiles/r01h) overlaps the next frame
    F = max(1, args.frames_in_flight)
    lanes = []
    for k in range(F):
        c = ctx if k == 0 else crt.Context(local)
        for k_, v_ in options:
            c.crt_set_option(k_, int(v_))
        md = mats_dev if k == 0 else c.upload(scene.materials)
        lanes.append({"ctx": c, "mats_dev": md, "mats": c.scene_mats(md, len(scene.materials), scene.env), "stream": torch.cuda.Stream(device=ctx.device)})

    def time_pipelined(mode):
        """W warm-up + K timed frames of one mode, frame i on lane i mod F (own context, stream, workspace, accumulation image)."""
        order = crt.make_order(mode, gw, gh, s)
        fr0 = crt.make_frame(w, h, spp)
        for ln in lanes:
            ln["ws"] = ln["ctx"].frame_workspace(fr0, order)
            ln["accum"] = torch.zeros((h, w, 3), device=ctx.device)
            ln["nsec"] = torch.zeros((K + W, max(nb, 1)), dtype=torch.int32, device=ctx.device)

        def step(i):
            ln = lanes[i % F]
            fr = crt.make_frame(w, h, spp, seed, replica_frame_index(i, rank, world))
            ln["ctx"].crt_render_frame(bvh, ln["mats"], cam, fr, order, nb, ln["accum"], ln["ws"], n_secondary=ln["nsec"][i], stream=ln["stream"])
        torch.cuda.synchronize()
        for i in range(W):
            step(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for ln in lanes:
            ln["stream"].wait_event(e0)
        for i in range(W, W + K):
            step(i)
        for ln in lanes:
            stream.wait_stream(ln["stream"])
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        rays = sum(int(ln["nsec"][W:].sum().item()) for ln in lanes)
        ms_all, rays_all = reduce_over_ranks(ms, rays, ctx.device, world)
        for ln in lanes:
            ln.pop("ws"); ln.pop("accum"); ln.pop("nsec")
        return {"mray_s": rays_all / (ms_all * 1e-3) / 1e6, "ms_per_step": ms_all / K, "frames_in_flight": F}

    def time_host_pipelined(mode):
        """The e2e leg with F host frames in flight: every step enqueues, on its lane's stream, the H2D copy of its inputs (materials,
        camera; pinned or staged by the runtime), the frame, and the D2H copy of the accumulated image and the ray counts into pinned
        host memory (crt_render_frame_host_resident_async); before a lane is reused its stream is synchronised, i.e. the host has its
        previous result.  The D2H copy of one frame overlaps the next frame's kernels."""
        order = crt.make_order(mode, gw, gh, s)
        fr0 = crt.make_frame(w, h, spp)
        for ln in lanes:
            ln["ws"] = ln["ctx"].frame_workspace(fr0, order, host_materials=len(scene.materials))
            ln["img_h"] = torch.zeros((h, w, 3), dtype=torch.float32).pin_memory()
            ln["nsec_h"] = torch.zeros((K + W, max(nb, 1)), dtype=torch.int32).pin_memory()
            ln["used"] = False

        def step(i):
            ln = lanes[i % F]
            if ln["used"]:
                ln["stream"].synchronize()
            fr = crt.make_frame(w, h, spp, seed, replica_frame_index(i, rank, world))
            ln["ctx"].crt_render_frame_host_resident(bvh, scene.materials, scene.env, cam, fr, order, nb, not ln["used"], ln["img_h"], ln["nsec_h"][i], ln["ws"],
                                                     stream=ln["stream"], wait=False)
            ln["used"] = True
        torch.cuda.synchronize()
        for i in range(W):
            step(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for ln in lanes:
            ln["stream"].wait_event(e0)
        for i in range(W, W + K):
            step(i)
        for ln in lanes:
            stream.wait_stream(ln["stream"])
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        rays = sum(int(ln["nsec_h"][W:].sum().item()) for ln in lanes)
        ms_all, rays_all = reduce_over_ranks(ms, rays, ctx.device, world)
        # each lane accumulates every F-th frame in its own resident image; the image a consumer shows is their sum over the frame count
        # (one host add per DISPLAYED image, not per step: done here once, outside the timed region)
        total = sum(ln["img_h"].double() for ln in lanes) / (K + W)
        img_mean = float(total.mean().item())
        for ln in lanes:
            for k in ("ws", "img_h", "nsec_h", "used"):
                ln.pop(k)
        return {"mray_s": rays_all / (ms_all * 1e-3) / 1e6, "ms_per_step": ms_all / K, "mean_of_summed_lane_images": img_mean}

    clocks = ClockSampler(local)
    modes = {}
    clocks.start()
    modes["direct_reuse"] = time_mode("direct_reuse")
    modes["independent"] = time_mode("independent")
    modes["morton_reorder"] = time_mode("morton_reorder")
    if args.repeats > 1:       # BASELINE config 5 / "beats both baselines": spread over repeated passes of K steps, not one number
        for m in ("direct_reuse", "independent", "morton_reorder"):
            runs = [modes[m]] + [time_mode(m) for _ in range(args.repeats - 1)]
            modes[m]["repeats"] = {k: {"min": float(np.min([r[k] for r in runs])), "median": float(np.median([r[k] for r in runs])), "max": float(np.max([r[k] for r in runs])), "n": len(runs)}
                                   for k in ("mray_s", "secondary_loop_mray_s", "trace_only_mray_s", "ms_per_step")}
    modes["world_reuse"] = time_mode("world_reuse")       # the paper's first variant, an ablation: biased, see DESIGN.md D:R18
    if not args.no_sort_codes:                            # the paper's other reordering baselines (Table 1; D:R19)
        for m in ("sort_origin", "sort_reis", "sort_costa", "sort_twopoint"):
            modes[m] = time_mode(m)
    single = time_mode("direct_reuse", stages=False)       # one frame at a time as a user calls it: no per-stage events, frame in bands
    e2e_one = time_mode("direct_reuse", host=True)
    e2e = time_host_pipelined("direct_reuse") if F > 1 else e2e_one
    piped = {m: time_pipelined(m) for m in ("direct_reuse", "independent", "morton_reorder")} if F > 1 else {}
    for m, v in piped.items():
        modes[m]["pipelined_mray_s"] = v["mray_s"]; modes[m]["pipelined_ms_per_step"] = v["ms_per_step"]
    clk = clocks.stop()

    # ---- roofline of the dominant kernel (secondary crt_trace): work counters of one frame's secondary rays, outside the timed region
    order = crt.make_order("direct_reuse", gw, gh, s)
    fr = crt.make_frame(w, h, spp, seed, W * world + rank)
    rays, hits, r2p = ctx.crt_trace_primary(bvh, cam, fr, order)
    n_paths = crt.crt_layout(fr, order)[0]
    paths = ctx.empty((n_paths, 8)); ctx.crt_paths_init(paths)
    acc = torch.zeros((h, w, 3), device=ctx.device)
    ctx.crt_shade_accumulate(bvh, mats, fr, 0, nb == 0, rays, hits, r2p, paths, acc)
    nn = nt = act = 0
    for b in range(1, nb + 1):
        out = ctx.crt_generate_secondary(bvh, mats, fr, b, order, rays, hits, r2p, paths)
        rays, r2p = out["rays"], out["ray_to_path"]
        c = ctx.crt_trace_stats(bvh, rays)
        nn += c[0]; nt += c[1]; act += c[2]
        hits = ctx.crt_trace(bvh, rays)
        ctx.crt_shade_accumulate(bvh, mats, fr, b, b == nb, rays, hits, r2p, paths, acc)
    launches = max(nb, 1)
    rays_per_launch = act / launches
    dr = modes["direct_reuse"]
    flop_per_ray_model = (nn * FLOP_PER_NODE_VISIT + nt * FLOP_PER_TRI_TEST + act * FLOP_PER_RAY) / max(act, 1)
    ncu = NCU_PER_RAY.get(args.workload) or {}
    flop_per_ray = ncu.get("flop") or flop_per_ray_model            # the ncu count when a profile of this workload exists
    ffma_tflops, copy_gbs = ctx.crt_measure_peaks()                  # FP32 peak: FFMA loop measured in THIS run (north_star: "measured")
    hbm_gbs, hbm_src = _peaks()
    achieved = flop_per_ray * rays_per_launch / (dr["trace_launch_ms"] * 1e-3) / 1e12
    traffic = ncu["dram_bytes"] * rays_per_launch if ncu.get("dram_bytes") else None
    bound_alu = ffma_tflops * 1e12 / flop_per_ray / 1e6             # MRay/s
    bound_hbm = (hbm_gbs * 1e9 / ncu["dram_bytes"] / 1e6) if ncu.get("dram_bytes") else None
    roofline = {"bound": "alu", "kernel": "trace_dyn_kernel<0,1> (crt_trace: 16-bit nodes, packed FFMA2; secondary rays in direct_reuse order)", "achieved": achieved,
                "peak": ffma_tflops, "unit": "TFLOP/s", "frac": achieved / ffma_tflops, "traffic": traffic,
                "peak_source": "FFMA loop measured in this run (crt_measure_peaks); nominal 148 SM x 128 lanes x 2 x 1.965 GHz = %.2f TFLOP/s" % FP32_PEAK_TFLOPS_NOMINAL,
                "flop_per_ray": flop_per_ray, "flop_per_ray_source": ncu.get("source") or "model (no ncu profile of this workload)",
                "flop_per_ray_model": flop_per_ray_model, "frac_model_flops_nominal_peak": flop_per_ray_model * rays_per_launch / (dr["trace_launch_ms"] * 1e-3) / 1e12 / FP32_PEAK_TFLOPS_NOMINAL,
                "dram_bytes_per_ray": ncu.get("dram_bytes"), "node_visits_per_ray": nn / max(act, 1), "tri_tests_per_ray": nt / max(act, 1),
                "rays_per_launch": rays_per_launch, "launch_ms": dr["trace_launch_ms"],
                "mray_s_bound_alu": bound_alu, "mray_s_bound_hbm": bound_hbm, "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": hbm_src,
                "copy_gbs_this_run": copy_gbs, "frac_of_min_bound": dr["trace_only_mray_s"] / min(bound_alu, bound_hbm or bound_alu),
                "limiter": TRACE_LIMITER.get(args.workload)}

    if rank != 0:
        return
    cpu = cpu_baseline(args.workload) if world == 1 and not args.no_cpu_baseline else None
    ws_bytes = int(crt.lib().crt_frame_workspace_bytes(__import__("ctypes").byref(fr), __import__("ctypes").byref(order)))
    img_bytes = w * h * 12
    head = piped["direct_reuse"] if F > 1 else dr          # headline: whole-step throughput with F frames in flight
    line = {
        "metric": METRIC, "value": head["mray_s"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": head["ms_per_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE config {cfg + 1}: {args.workload} scene, {info['n_tris']} triangles, {w}x{h}, {spp} spp, {nb} bounces, "
                               f"direct_reuse groups {gw}x{gh} stride {s}, seed {seed}",
                   "mode": "direct_reuse", "value_is": "live secondary rays per step / device time of the whole step (primary + shading included)",
                   "frames_in_flight": F, "single_stream_value": single["mray_s"], "single_stream_ms_per_step": single["ms_per_step"],
                   "single_stream_note": "one frame at a time without per-stage events (crt_render_frame then cuts the frame into bands, option frame_bands); modes[..].mray_s are with per-stage events, unbanded",
                   "l2": f"no explicit flush: each step streams its {ws_bytes / 1e6:.0f} MB workspace plus the {info['device_bytes'] / 1e6:.0f} MB BVH (> 126 MB L2)",
                   "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
                   "bvh": {"nodes": info["n_nodes"], "triangle_references": info["n_refs"], "presplit": BVH_KW.get("presplit", "library default (1/16 of the scene diagonal)"), "optimize": BVH_KW.get("optimize", "library default (20 iterations)"), "depth": info["depth"], "sah_cost": info["sah_cost"], "device_mb": info["device_bytes"] / 1e6,
                           "build_s": info["build_seconds"], "build_and_upload_s": build_s}},
        "modes": modes, "roofline": roofline, "cpu_baseline": cpu,
        "e2e": {"value": e2e["mray_s"], "unit": UNIT, "h2d_bytes_per_step": len(scene.materials) * 32 + 48 + 24,
                "d2h_bytes_per_step": img_bytes + 4 * nb, "ms_per_step": e2e["ms_per_step"],
                "api": "crt_render_frame_host_resident_async, %d host frames in flight" % F if F > 1 else "crt_render_frame_host_resident",
                "one_frame_at_a_time": e2e_one["mray_s"],
                "image": "each lane keeps a resident accumulation image and copies its sum so far out every step; displayed image = sum of the lane images / frames (mean radiance %.6f)" % e2e.get("mean_of_summed_lane_images", float("nan"))},
        # kernels of the K timed steps of the headline pass: primary_rays, trace, then per bounce generate (with the previous segment's
        # shading and, at the first bounce, the initial path state fused in: the library's default) + trace, then the final shade
        "gpu_launches": K * ((3 + 2 * nb) if nb >= 1 else 4), "clocks": clk,
    }
    print(json.dumps(line))


def run_sweep(args):
    """BASELINE config 3: interior scene at 3840x2160, 4 spp, 3 bounces; group size {2,4,8}^2 x stride {1,2,4,8} plus independent.
    Per point: secondary MRay/s over `--sweep-frames` frames and the RMSE of their mean image against (a) the mean of the same number
    of independent-sampling frames and (b) a longer independent reference (--sweep-reference-frames; default 4x the frames).  One JSON line ("sweep": [...]).
    Warp execution efficiency and L2 hit rate come from ncu (profiles/), not from this run."""
    import torch
    import paper_2310_07182_b200 as crt
    ctx = crt.Context(0)
    import crt_inputs as I
    sc = max(1, args.sweep_scale)
    table3 = args.sweep == "table3"
    rules = args.sweep == "rules"
    w, h, spp, nb, seed = (1920 // sc, 1080 // sc, 1, 2, 1) if (table3 or rules or args.sweep == "bias") else (3840 // sc, 2160 // sc, 4, 3, 1)
    bias_cornell = args.sweep == "bias" and args.workload == "cornell"      # the all-Lambert scene: every group is a DIFFUSE group
    if bias_cornell:
        w, h, nb = 512, 512, 2
    scene = (I.by_name("cornell") if bias_cornell else I.by_name("interior", seed=1)).with_camera(w, h)
    if args.sweep == "bias" and args.all_lambert:      # the same geometry with every glossy and mirror material made Lambert: no GLOSSY or HYBRID group is left
        t = scene.materials["type"]; t[(t == I.scenes.MAT_GLOSSY) | (t == I.scenes.MAT_SPECULAR)] = I.scenes.MAT_DIFFUSE
    bvh = ctx.crt_build_bvh(scene.verts, scene.mat_id, **BVH_KW)
    mats_dev = ctx.upload(scene.materials); mats = ctx.scene_mats(mats_dev, len(scene.materials), scene.env)
    cam = crt.make_camera(scene.camera)
    F = args.sweep_frames

    def render(mode, g, s, frames, first_frame, tile=None, rule=0):
        order = crt.order_for_tile(mode, *tile) if tile else crt.make_order(mode, g, g, s, partition_rule=rule)
        fr0 = crt.make_frame(w, h, spp)
        ws = ctx.frame_workspace(fr0, order)
        accum = torch.zeros((h, w, 3), device=ctx.device)
        nsec = torch.zeros((frames, nb), dtype=torch.int32, device=ctx.device)
        stage = np.zeros(8, np.float32)
        for i in range(2):                                        # warm-up on frames outside the accumulated range
            ctx.crt_render_frame(bvh, mats, cam, crt.make_frame(w, h, spp, seed, 1000000 + i), order, nb, torch.zeros_like(accum), ws)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); e0.record()
        for i in range(frames):
            ctx.crt_render_frame(bvh, mats, cam, crt.make_frame(w, h, spp, seed, first_frame + i), order, nb, accum, ws, n_secondary=nsec[i], record_times=True)
            ctx.crt_frame_times(stage)
        e1.record(); torch.cuda.synchronize()
        rays = int(nsec.sum().item()); ms = e0.elapsed_time(e1)
        del ws
        return accum / frames, {"mray_s": rays / (ms * 1e-3) / 1e6, "secondary_loop_mray_s": rays / (float(stage[2] + stage[3]) * 1e-3) / 1e6,
                                "trace_only_mray_s": rays / (float(stage[3]) * 1e-3) / 1e6, "ms_per_frame": ms / frames}

    def rmse(a, b):
        return float(torch.sqrt(torch.mean((a.double() - b.double()) ** 2)).item())

    if args.sweep == "bias":
        # Does the mean image of a reuse mode converge to independent sampling's?  (sharing a WORLD direction skews the members' distributions --
        # the paper's Fig. 1 artefacts --, sharing the LOCAL direction does not; HYBRID groups' averaged direction is a heuristic.)  Four F-frame means at
        # BASELINE config 2's size: independent over two disjoint frame ranges (their RMSE is the noise floor), direct_reuse and world_reuse over a third.
        ind_a, _ = render("independent", 1, 1, F, 0)
        ind_b, _ = render("independent", 1, 1, F, 500000)
        out = {"noise_floor_rmse_independent_vs_independent": rmse(ind_a, ind_b)}
        for mode in ("direct_reuse", "world_reuse"):
            for g, st in ((4, 4), (8, 1)):
                img, _ = render(mode, g, st, F, 1000000)
                out[f"{mode}_{g}x{g}_stride{st}"] = {"rmse_vs_independent": rmse(img, ind_b), "mean_image": float(img.mean().item()), "mean_independent": float(ind_b.mean().item())}
        print(json.dumps({"clocks": _SWEEP_CLOCKS.stop() if _SWEEP_CLOCKS else None, "bias": out, "config": {"workload": f"{'cornell (all Lambert)' if bias_cornell else 'interior'} scene {w}x{h}, {spp} spp, {nb} bounces", "all_lambert": bool(args.all_lambert), "frames_per_mean": F}}))
        return
    RF = args.sweep_reference_frames or 4 * F
    ref, _ = render("independent", 1, 1, RF, 500000)              # disjoint frame range: independent of every sweep point
    ind, ind_t = render("independent", 1, 1, F, 0)
    points = [dict(mode="independent", group=1, stride=1, **ind_t, rmse_vs_reference=rmse(ind, ref), rmse_vs_independent=0.0)]
    if table3:      # P:L178-185 (Table 3): tile (8,8), (16,8), (16,16), (32,8) x K = 8, 16, 32, 64
        for tw, th in ((8, 8), (16, 8), (16, 16), (32, 8)):
            for k in (8, 16, 32, 64):
                img, t = render("direct_reuse", 0, 0, F, 0, tile=(tw, th, k))
                points.append(dict(mode="direct_reuse", tile=[tw, th], K=k, **t, rmse_vs_reference=rmse(img, ref), rmse_vs_independent=rmse(img, ind),
                                   trace_speedup_vs_independent=t["trace_only_mray_s"] / ind_t["trace_only_mray_s"]))
    elif rules:     # the three partition rules side by side (DESIGN.md D:R3 affine shuffle, D:R20 regular lattice, D:R21 LCG sequence)
        for g in (4, 8):
            for s in (2, 4, 8):
                for rule, rname in ((0, "shuffle"), (1, "lattice"), (2, "lcg_sequence")):
                    img, t = render("direct_reuse", g, s, F, 0, rule=rule)
                    points.append(dict(mode="direct_reuse", group=g, stride=s, partition_rule=rname, **t, rmse_vs_reference=rmse(img, ref), rmse_vs_independent=rmse(img, ind),
                                       trace_speedup_vs_independent=t["trace_only_mray_s"] / ind_t["trace_only_mray_s"]))
    else:
        for g in (2, 4, 8):
            for s in (1, 2, 4, 8):
                img, t = render("direct_reuse", g, s, F, 0)
                points.append(dict(mode="direct_reuse", group=g, stride=s, **t, rmse_vs_reference=rmse(img, ref), rmse_vs_independent=rmse(img, ind)))
    name = "the paper's Table 3 shapes (P:L178-185)" if table3 else ("partition rules (D:R3 / D:R20 / D:R21)" if rules else "BASELINE config 3")
    print(json.dumps({"clocks": _SWEEP_CLOCKS.stop() if _SWEEP_CLOCKS else None, "sweep": points, "config": {"workload": f"{name}: interior scene {w}x{h}, {spp} spp, {nb} bounces", "frames": F,
                                                  "reference_frames": RF, "scale": sc}}))


def _frame_ray_sets(ctx, crt, scene, w, h, spp, nb, gw, gh, s, seed, frame, modes=("direct_reuse", "independent"), bvh=None):
    """The ray sets of one frame (primary, bounce 1 .. nb) in each order of `modes`: [(tag, rays)]."""
    import torch
    bvh = bvh or ctx.crt_build_bvh(scene.verts, scene.mat_id, **BVH_KW)
    mats_dev = ctx.upload(scene.materials); mats = ctx.scene_mats(mats_dev, len(scene.materials), scene.env); cam = crt.make_camera(scene.camera)
    sets = []
    for mode in modes:
        order = crt.make_order(mode, gw, gh, s) if mode == "direct_reuse" else crt.make_order(mode)
        fr = crt.make_frame(w, h, spp, seed, frame)
        rays, hits, r2p = ctx.crt_trace_primary(bvh, cam, fr, order)
        paths = ctx.empty((crt.crt_layout(fr, order)[0], 8)); ctx.crt_paths_init(paths)
        acc = torch.zeros((h, w, 3), device=ctx.device)
        ctx.crt_shade_accumulate(bvh, mats, fr, 0, False, rays, hits, r2p, paths, acc)
        sets.append((f"{mode} primary", rays.clone()))
        for b in range(1, nb + 1):
            out = ctx.crt_generate_secondary(bvh, mats, fr, b, order, rays, hits, r2p, paths)
            rays, r2p = out["rays"], out["ray_to_path"]
            sets.append((f"{mode} bounce {b}", rays.clone()))
            hits = ctx.crt_trace(bvh, rays)
            ctx.crt_shade_accumulate(bvh, mats, fr, b, b == nb, rays, hits, r2p, paths, acc)
    return bvh, (mats_dev, mats), sets


BVH_KW = {}      # --presplit: build parameter of every BVH this run builds (default: the library's)
KERNEL_OPTION_DEFAULTS = {"trace_kernel": 3, "trace_refill_threshold": 16, "trace_leaf_wait": 6, "trace_blocks_per_sm": 0, "trace_exact": 1, "trace_tail_split": 0}


def run_kernels(args):
    """A/B of traversal kernel variants (profiles/r02a): crt_trace alone on the ray sets of one frame (frame 7; primary, bounce 1, bounce 2;
    direct_reuse and independent order), L2 flushed between repetitions, median of 8; hit records compared with the default kernel's.
    --variants: comma-free list like "3 5 6 3:trace_exact=0 3:trace_blocks_per_sm=6" (trace_kernel id, then option=value pairs)."""
    import torch
    import paper_2310_07182_b200 as crt
    import crt_inputs as I
    name, kw, w, h, spp, nb, gw, gh, s, seed, cfg = WORKLOADS[args.workload]
    scene = I.by_name(name, **kw).with_camera(w, h)
    ctx = crt.Context(0)
    bvh, _keep, sets = _frame_ray_sets(ctx, crt, scene, w, h, spp, nb, gw, gh, s, seed, 7)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctx.device)
    ref = {tag: ctx.crt_trace(bvh, r).clone() for tag, r in sets}
    torch.cuda.synchronize()
    rows = []
    for v in args.variants:
        k, _, opts = v.partition(":")
        ctx.crt_set_option("trace_kernel", int(k))
        touched = []
        for o in filter(None, opts.split(",")):
            key, val = o.split("="); ctx.crt_set_option(key, int(val)); touched.append(key)
        row = {"variant": v, "sets": {}}
        for tag, r in sets:
            hh = ctx.crt_trace(bvh, r); torch.cuda.synchronize()
            hi, ri = hh.view(torch.int32), ref[tag].view(torch.int32)
            ids_equal = float((hi[:, 3] == ri[:, 3]).float().mean().item())
            ts = []
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(8):
                flush.fill_(1)
                e0.record(); ctx.crt_trace(bvh, r, hits=hh); e1.record(); torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            nv, nt, nr, npk = ctx.crt_trace_stats(bvh, r, full=True)
            row["sets"][tag] = {"ms": float(np.median(ts)), "records_identical": bool(torch.equal(hi, ri)), "ids_equal_frac": ids_equal, "active_rays": int(nr),
                                "node_visits_per_ray": nv / max(1, nr), "tri_tests_per_ray": nt / max(1, nr)}
            if npk:      # trace_kernel 8: node visits of a 16-ray packet, per ray of the packet (x 16 = lane slots issued per ray's share)
                row["sets"][tag]["packet_visits_per_16_rays"] = 16.0 * npk / max(1, nr)
        rows.append(row)
        for key in ["trace_kernel"] + touched:
            ctx.crt_set_option(key, KERNEL_OPTION_DEFAULTS[key])
    print(json.dumps({"clocks": _SWEEP_CLOCKS.stop() if _SWEEP_CLOCKS else None, "kernels": rows, "config": {"workload": args.workload, "order": f"direct_reuse {gw}x{gh} stride {s} / independent", "frame": 7,
                                                  "timing": "crt_trace alone, CUDA events, median of 8, 256 MB L2 flush between repetitions"}}))
    tags = [t for t, _ in sets]
    sys.stderr.write("| variant | " + " | ".join(tags) + " |\n|---|" + "---:|" * len(tags) + "\n")
    for row in rows:
        sys.stderr.write(f"| {row['variant']} | " + " | ".join(f"{row['sets'][t]['ms']:.3f}{'' if row['sets'][t]['records_identical'] else ' (ids ' + format(row['sets'][t]['ids_equal_frac'], '.6f') + ')'}" for t in tags) + " |\n")


def run_builders(args):
    """Host (binned SAH) against device (PLOC, csrc/bvh_ploc.cu) BVH builder on --workload (profiles/r02b): build times, tree statistics,
    crt_bvh_check, and crt_trace on one frame's ray sets (as --sweep kernels) with each tree; hit records must be identical."""
    import torch
    import paper_2310_07182_b200 as crt
    import crt_inputs as I
    name, kw, w, h, spp, nb, gw, gh, s, seed, cfg = WORKLOADS[args.workload]
    scene = I.by_name(name, **kw).with_camera(w, h)
    ctx = crt.Context(0)
    trees = []
    for label, bkw in [("host SAH + pre-split, re-insertion on the device (default)", dict(builder=0)), ("host SAH + pre-split, re-insertion on the host (builder 3)", dict(builder=3)), ("host SAH + pre-split, no optimisation", dict(builder=0, optimize=0))] + [(f"device PLOC radius {r}", dict(builder=1, ploc_radius=r, optimize=0)) for r in args.ploc_radii] + [(f"device PLOC radius {args.ploc_radii[0]} + device re-insertion", dict(builder=1, ploc_radius=args.ploc_radii[0]))] + [(f"device clustering radius {args.ploc_radii[0]} + host optimisation and layout", dict(builder=2, ploc_radius=args.ploc_radii[0]))]:
        t0 = time.time(); bvh = ctx.crt_build_bvh(scene.verts, scene.mat_id, **bkw); wall = time.time() - t0
        info = bvh.info()
        trees.append((label, bvh, dict(builder=label, wall_seconds=wall, hierarchy_seconds=info["build_seconds"], device_build_seconds=info["device_build_seconds"],
                                       layout_seconds=info["layout_seconds"], rounds=info["build_rounds"], optimize_iterations=info["optimize_iterations"], depth=info["depth"], sah_cost=info["sah_cost"],
                                       n_nodes=info["n_nodes"], q16_inflation_pct=info["q16_inflation_pct"], check=bvh.check())))
    _, _keep, sets = _frame_ray_sets(ctx, crt, scene, w, h, spp, nb, gw, gh, s, seed, 7, bvh=trees[0][1])
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctx.device)
    ref = {tag: ctx.crt_trace(trees[0][1], r).clone() for tag, r in sets}
    rows = []
    for label, bvh, row in trees:
        row["sets"] = {}
        for tag, r in sets:
            hh = ctx.crt_trace(bvh, r); torch.cuda.synchronize()
            ts = []
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(8):
                flush.fill_(1)
                e0.record(); ctx.crt_trace(bvh, r, hits=hh); e1.record(); torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            nv, nt, nr = ctx.crt_trace_stats(bvh, r)
            row["sets"][tag] = {"ms": float(np.median(ts)), "records_identical": bool(torch.equal(hh.view(torch.int32), ref[tag].view(torch.int32))),
                                "node_visits_per_ray": nv / max(1, nr), "tri_tests_per_ray": nt / max(1, nr)}
        rows.append(row)
    print(json.dumps({"clocks": _SWEEP_CLOCKS.stop() if _SWEEP_CLOCKS else None, "builders": rows, "config": {"workload": args.workload, "n_tris": int(scene.n_tris), "frame": 7,
                                                   "timing": "crt_trace alone, CUDA events, median of 8, 256 MB L2 flush between repetitions"}}))
    tags = [t for t, _ in sets]
    sys.stderr.write("| builder | hierarchy s | of which on device s | layout s | rounds | opt iterations | depth | SAH cost | check | " + " | ".join(tags) + " |\n|---|" + "---:|" * (8 + len(tags)) + "\n")
    for row in rows:
        sys.stderr.write(f"| {row['builder']} | {row['hierarchy_seconds']:.3f} | {row['device_build_seconds']:.4f} | {row['layout_seconds']:.3f} | {row['rounds']} | {row['optimize_iterations']} | {row['depth']} | {row['sah_cost']:.1f} | {row['check']} | "
                         + " | ".join(f"{row['sets'][t]['ms']:.3f}{'' if row['sets'][t]['records_identical'] else ' !'}" for t in tags) + " |\n")


def run_timeline(args):
    """What the tail of a persistent crt_trace launch consists of (profiles/r02i): crt_trace_timeline (the default kernel with four time marks
    per warp) on the three direct_reuse ray sets of one frame of --workload, with and without trace_tail_split; L2 flushed, third repetition.
    All times in microseconds after the first warp's start.  One JSON line."""
    import torch
    import paper_2310_07182_b200 as crt
    import crt_inputs as I
    name, kw, w, h, spp, nb, gw, gh, s, seed, cfg = WORKLOADS[args.workload]
    scene = I.by_name(name, **kw).with_camera(w, h)
    ctx = crt.Context(0)
    bvh, _keep, sets = _frame_ray_sets(ctx, crt, scene, w, h, spp, nb, gw, gh, s, seed, 7)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctx.device)
    rows = []
    for split in (0, 1):
        ctx.crt_set_option("trace_tail_split", split)
        for tag, r in sets[:3]:
            ref = ctx.crt_trace(bvh, r).clone()
            for _ in range(3):
                flush.fill_(1); hh, marks = ctx.crt_trace_timeline(bvh, r); torch.cuda.synchronize()
            t0 = marks[:, 0].min()
            start, exh, end = (marks[:, 0] - t0) / 1e3, (marks[:, 1] - t0) / 1e3, (marks[:, 2] - t0) / 1e3
            seen = marks[:, 1] > 0
            first_exh = float(exh[seen].min()) if seen.any() else float("nan")
            rows.append({"tail_split": split, "set": tag, "warps": int(marks.shape[0]), "records_identical": bool(torch.equal(hh.view(torch.int32), ref.view(torch.int32))),
                         "span_us": float(end.max()), "last_warp_start_us": float(start.max()), "ray_list_exhausted_first_seen_us": first_exh, "last_seen_us": float(exh[seen].max()) if seen.any() else float("nan"),
                         "warp_end_us_p10_p50_p90_p99_max": [float(np.percentile(end, q)) for q in (10, 50, 90, 99, 100)],
                         "tail_us": float(end.max()) - first_exh,
                         "lane_visits_after_exhaustion_p50_p90_max": [float(np.percentile(marks[:, 3], 50)), float(np.percentile(marks[:, 3], 90)), float(marks[:, 3].max())]})
    ctx.crt_set_option("trace_tail_split", KERNEL_OPTION_DEFAULTS["trace_tail_split"])
    print(json.dumps({"clocks": _SWEEP_CLOCKS.stop() if _SWEEP_CLOCKS else None, "timeline": rows, "config": {"workload": args.workload, "order": f"direct_reuse {gw}x{gh} stride {s}", "frame": 7,
                                                   "timing": "per-warp %globaltimer marks inside the kernel (crt_trace_timeline), third repetition, 256 MB L2 flush before each"}}))
    for row in rows:
        sys.stderr.write(f"split {row['tail_split']} {row['set']}: span {row['span_us']:.1f} us, list exhausted at {row['ray_list_exhausted_first_seen_us']:.1f}, warp ends p10/p50/p90/p99/max "
                         + "/".join(f"{x:.1f}" for x in row["warp_end_us_p10_p50_p90_p99_max"]) + f", tail {row['tail_us']:.1f} us, visits after exhaustion p50/p90/max " + "/".join(f"{x:.0f}" for x in row["lane_visits_after_exhaustion_p50_p90_max"]) + "\n")


def run_tail(args):
    """Fixed cost of a crt_trace launch (profiles/r01h): crt_trace on one frame's ray sets (primary, bounce 1, bounce 2; direct_reuse order)
    and on the same set concatenated twice and four times; L2 flushed between repetitions, median of 8.  One JSON line."""
    import torch
    import paper_2310_07182_b200 as crt
    import crt_inputs as I
    name, kw, w, h, spp, nb, gw, gh, s, seed, cfg = WORKLOADS[args.workload]
    scene = I.by_name(name, **kw).with_camera(w, h)
    ctx = crt.Context(0)
    bvh = ctx.crt_build_bvh(scene.verts, scene.mat_id, **BVH_KW)
    mats_dev = ctx.upload(scene.materials); mats = ctx.scene_mats(mats_dev, len(scene.materials), scene.env); cam = crt.make_camera(scene.camera)
    order = crt.make_order("direct_reuse", gw, gh, s); fr = crt.make_frame(w, h, spp, seed, 7)
    rays, hits, r2p = ctx.crt_trace_primary(bvh, cam, fr, order)
    paths = ctx.empty((crt.crt_layout(fr, order)[0], 8)); ctx.crt_paths_init(paths)
    acc = torch.zeros((h, w, 3), device=ctx.device)
    ctx.crt_shade_accumulate(bvh, mats, fr, 0, False, rays, hits, r2p, paths, acc)
    sets = [("primary", rays.clone())]
    for b in range(1, nb + 1):
        out = ctx.crt_generate_secondary(bvh, mats, fr, b, order, rays, hits, r2p, paths)
        rays, r2p = out["rays"], out["ray_to_path"]
        sets.append((f"bounce {b}", rays.clone()))
        hits = ctx.crt_trace(bvh, rays)
        ctx.crt_shade_accumulate(bvh, mats, fr, b, b == nb, rays, hits, r2p, paths, acc)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctx.device)

    def t_trace(r):
        hh = ctx.crt_trace(bvh, r); ts = []
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(8):
            flush.fill_(1)
            e0.record(); ctx.crt_trace(bvh, r, hits=hh); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))
    rows = []
    for tag, r in sets:
        t1 = t_trace(r); r2 = torch.cat([r, r]).contiguous(); t2 = t_trace(r2); t4 = t_trace(torch.cat([r2, r2]).contiguous())
        rows.append({"rays": tag, "n": int(r.shape[0]), "t_n_ms": t1, "t_2n_ms": t2, "t_4n_ms": t4, "fixed_ms_from_2n": 2 * t1 - t2, "fixed_ms_from_4n": (4 * t1 - t4) / 3})
    print(json.dumps({"clocks": _SWEEP_CLOCKS.stop() if _SWEEP_CLOCKS else None, "tail": rows, "config": {"workload": args.workload, "order": f"direct_reuse {gw}x{gh} stride {s}", "frame": 7}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)      # the paper averages 100 frames per run
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="interior", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--frames-in-flight", type=int, default=3, help="frames rendered concurrently (one context + stream each) for the headline value; the per-mode table stays single-stream")
    ap.add_argument("--set", nargs="*", default=[], metavar="OPTION=VALUE", help="crt_set_option on every context of the run (experiments; the defaults are what the driver times)")
    ap.add_argument("--repeats", type=int, default=1, help="repeat the K timed steps of direct_reuse / independent / morton_reorder this many times and report min / median / max")
    ap.add_argument("--no-sort-codes", action="store_true", help="skip the Origin / Reis / Costa / TwoPoint reordering baselines")
    ap.add_argument("--sweep", nargs="?", const="config3", default=None, choices=["config3", "table3", "rules", "tail", "kernels", "builders", "timeline", "bias"],
                    help="config3: BASELINE config 3 sweep; table3: the paper's Table 3 shapes (tile x K) at 1920x1080, 1 spp, 2 bounces; rules: shuffled against lattice partition at the same size; tail: fixed cost of a crt_trace launch (n, 2n, 4n rays) on --workload; kernels: A/B of traversal kernel variants (--variants) on one frame's ray sets of --workload; timeline: per-warp time marks of a crt_trace launch (what its tail consists of); bias: long-run mean images of direct_reuse and world_reuse against independent sampling; builders: host SAH against device PLOC BVH builder on --workload")
    ap.add_argument("--ploc-radii", nargs="*", type=int, default=[8], help="--sweep builders: neighbour radii of the device builder")
    ap.add_argument("--variants", nargs="*", default=["3", "3:trace_exact=0", "5", "6", "4", "1"], help="--sweep kernels: trace_kernel id[:option=value,...] ...")
    ap.add_argument("--presplit", type=float, default=None, help="crt_bvh_params.presplit of the BVHs built by this run (0 = no pre-splitting of large triangles; default: the library's 1/16)")
    ap.add_argument("--bvh-optimize", type=int, default=None, help="crt_bvh_params.optimize of the BVHs built by this run (iterations of insertion-based tree optimisation; default: the library's 20)")
    ap.add_argument("--sweep-frames", type=int, default=64)
    ap.add_argument("--all-lambert", action="store_true", help="--sweep bias: turn every glossy / mirror material of the scene into a Lambert one")
    ap.add_argument("--sweep-reference-frames", type=int, default=0, help="frames of the independent-sampling reference image of a sweep (0 = 4 x --sweep-frames)")
    ap.add_argument("--sweep-scale", type=int, default=1, help="divide the 3840x2160 image by this (quick runs)")
    args = ap.parse_args()
    if args.presplit is not None:
        BVH_KW["presplit"] = args.presplit
    if args.bvh_optimize is not None:
        BVH_KW["optimize"] = args.bvh_optimize
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    if args.sweep:
        global _SWEEP_CLOCKS
        _SWEEP_CLOCKS = ClockSampler(0); _SWEEP_CLOCKS.start()       # every sweep line carries the clocks sampled during it
    if args.sweep == "tail":
        run_tail(args)
        return
    if args.sweep == "kernels":
        run_kernels(args)
        return
    if args.sweep == "timeline":
        run_timeline(args)
        return
    if args.sweep == "builders":
        run_builders(args)
        return
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
