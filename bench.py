#!/usr/bin/env python
"""bench.py -- ms per fwd+bwd raster step on the paper-shaped workload (BASELINE.json configs[2]: 1600x1200, 1 M surfels).

A "step" is one pass of the whole hot path over one view: ocgs_preprocess -> ocgs_bin_sort -> ocgs_render_fwd (background
loss L_b and visibility statistics on, with the harness masked-L1 term of S20 fused: ocgs_render_fwd_l1) -> ocgs_render_bwd, all
through the C ABI.  Views rotate over a fixed set; inputs are resident in HBM before the timed region (`value`), or in
pinned host memory with the copies inside the timed region (`e2e`, through ocgs_step_view_host).  `--impl reference` times the
CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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
sys.path.insert(0, ROOT)

METRIC = "ms per fwd+bwd raster step (1600x1200, 1M surfels)"
FLOP_EVAL, FLOP_BLEND_FWD, FLOP_BLEND_BWD = 40.0, 22.0, 72.0  # DESIGN.md section 6 "algorithmic work per unit" (FMA = 2)
FLOP_BLEND_BWD_COLOUR_ONLY = 54.0  # no upstream gradient on depth / normal maps (masked L1 + L_b): those terms are not evaluated
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the raster kernels (bytes), from the `ncu --set full` capture of
# this workload committed under profiles/ (NCU_TRAFFIC_SOURCE)
NCU_TRAFFIC = {"render_bwd_kernel": 86.28e6, "render_fwd_kernel": 133.83e6}  # dram read + write of the two ordinary launches
NCU_TRAFFIC_SOURCE = "profiles/r02b_config3_raster_kernels_full.md"
# fallback only (used when the microbenchmark of ocgs_peak_probe cannot run): 148 SMs x 128 FP32 lanes x 2 (FMA) x max SM clock
ALU_PEAK_TFLOPS_DERIVED = 148 * 128 * 2 * 1.965e9 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="config3")
    ap.add_argument("--views", type=int, default=8, help="distinct views rotated over per rank (0 = the rank's whole shard of the config's views)")
    ap.add_argument("--batch-views", action="store_true",
                    help="N > 1 only: the N views of a step form one optimiser batch -- every step ends with the all-reduce (sum) of the gradient "
                         "arrays over ranks (SURVEY.md 8(e)); direct launches, the collective is inside the timed region")
    ap.add_argument("--shrink", type=float, default=1.0, help="scale surfel counts (debug only; invalidates the metric)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--loss", default="l1", choices=["l1", "dssim", "eq3"],
                    help="loss of the step: masked L1 (harness loss S20, the default the metric is quoted on); the full L_c^M = 0.8 L1 + 0.2 D-SSIM of "
                         "Eq. 2 (ocgs_photometric_loss); or all of Eq. 3 (moment forward, ocgs_regularizers, moment backward)")
    ap.add_argument("--no-prune", action="store_true", help="skip the separately timed prune pass (profiling runs)")
    ap.add_argument("--no-graph", action="store_true", help="time direct kernel launches instead of CUDA graph replays")
    return ap.parse_args()


def workload_name(scene):
    """The same string in both arms, so that the driver sees one config."""
    c = scene.cameras[0]
    return f"{scene.name}: {scene.n} surfels, {c.width}x{c.height}, SH degree {scene.sh_degree}, {len(scene.cameras)} views"


def make_scene(args):
    from paper_2501_08174_b200 import scenegen as sg
    kw = {}
    if args.shrink != 1.0:
        import inspect
        sig = inspect.signature(sg.CONFIGS[args.config]).parameters
        for k in ("n_obj", "n_bg", "n_shell", "n_in"):
            if k in sig:
                kw[k] = max(1, int(sig[k].default * args.shrink))
    return sg.make_scene(args.config, **kw)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f).get("hbm_gbs", 6650.0), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except ValueError:
                continue
            for nme, val in zip(names, f[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------------------------------

def oracle_sample(scene, view, window_frac=0.2):
    """One bounded sample of the step on the host cores: full preprocess + bin_sort of the view, forward and backward
    of a centred window of window_frac x window_frac of the image, extrapolated by pixel count.  Returns (ms per step
    extrapolated, description, cores)."""
    import oracle as orc
    cam_np = scene.cameras[view]
    cam = orc.camera_from(cam_np)
    cfg = orc.default_config(sh_degree=scene.sh_degree)
    W, H = cam_np.width, cam_np.height
    ww, wh = max(16, int(W * window_frac) // 16 * 16), max(16, int(H * window_frac) // 16 * 16)
    x0, y0 = (W - ww) // 2 // 16 * 16, (H - wh) // 2 // 16 * 16
    win = (x0, y0, x0 + ww, y0 + wh)
    mask = scene.mask(view)
    P = (scene.pos, scene.scale, scene.quat, scene.opacity, scene.sh)
    t0 = time.perf_counter()
    pre = orc.preprocess(*P, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    t1 = time.perf_counter()
    fwd = orc.render_fwd(pre, srt, scene.opacity, cam, cfg, mask=mask, window=win, want_fragile=False)
    gC = np.where(mask[None] > 0, np.sign(fwd["color"] - 0.5), 0.0) / (3.0 * W * H)
    orc.render_bwd(*P, pre, srt, cam, cfg, mask=mask, gC=gC, window=win)
    t2 = time.perf_counter()
    scale = (W * H) / float(ww * wh)
    ms = ((t1 - t0) + (t2 - t1) * scale) * 1e3
    desc = (f"view {view}: preprocess+bin_sort of all {scene.n} surfels ({(t1 - t0):.2f} s) + fwd+bwd of a centred {ww}x{wh} window "
            f"({(t2 - t1):.2f} s) scaled by {scale:.1f} to {W}x{H}")
    return ms, desc, orc.num_threads(), t2 - t1


def alu_peaks(B, torch, dev):
    """FP32-FMA and MUFU.EX2 rates of this device, measured with the library's microbenchmark (ocgs_peak_probe): best of five
    launches of ~1 ms, CUDA events on the launching stream.  SURVEY.md 8(d): the rooflines of the raster kernels are quoted
    against THESE, not against unit counts x clock."""
    props = torch.cuda.get_device_properties(dev)
    out = torch.empty(props.multi_processor_count * 8 * 256, dtype=torch.float32, device=dev)
    res = {}
    # kind 0: scalar FFMA with uniform (constant) b, c -- THE peak the rooflines are quoted against; 2: scalar FFMA with three register
    # operands, the form real kernels issue (register-file bound: measured 48 TFLOP/s); 3 / 4: packed fma.rn.f32x2 (FFMA2) with b, c
    # as broadcast scalars / as full register pairs
    for kind, key in ((0, "fp32_tflops_measured"), (1, "ex2_tops_measured"), (2, "fp32_tflops_3reg_measured"), (3, "fp32x2_bcast_tflops_measured"),
                      (4, "fp32x2_pairs_tflops_measured")):
        iters = 256 if kind == 1 else 2048  # ~1 ms per launch for every kind (EX2 issues at 1/16 of the FMA rate)
        best = 0.0
        for rep_i in range(13):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ops = B.ocgs_peak_probe(kind, iters, out)
            e1.record()
            torch.cuda.synchronize()
            if rep_i >= 3:  # the first launches warm up (clocks, instruction cache)
                best = max(best, ops / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        res[key] = best
    res["how"] = ("ocgs_peak_probe: 8 independent chains per thread of a <- fma(a,b,c) (2 flop; b, c uniform = fp32_tflops_measured, the roofline "
                  "peak; b, c in registers = fp32_tflops_3reg_measured; packed fma.rn.f32x2 with b, c broadcast scalars / full pairs = fp32x2_bcast_ / fp32x2_pairs_tflops_measured) / a <- -ex2(a), "
                  "8 blocks x 256 threads per SM, best of 10 launches after 3 warm-up launches, CUDA events")
    res["sm_count"] = props.multi_processor_count
    res["fp32_tflops_derived"] = ALU_PEAK_TFLOPS_DERIVED
    return res


def oracle_cores():
    """(threads the oracle uses, affinity mask of this process as a sorted list of CPU ids, os.cpu_count())"""
    import oracle as orc
    try:
        aff = sorted(os.sched_getaffinity(0))
    except AttributeError:
        aff = []
    return orc.num_threads(), aff, os.cpu_count()


def pick_window_frac(scene, view, budget_s):
    """Largest centred window (up to the whole image) whose forward + backward stays near budget_s of CPU work: the less is
    extrapolated the better -- a small window has too few tiles to keep all cores busy and sits on the object, which
    overstates the full step (measured: 15.6 s extrapolated from 160x112 against 4.8 s for the whole 1600x1200 view).
    Returns (fraction, last sample)."""
    frac, sample = 0.1, None
    for _ in range(3):
        sample = oracle_sample(scene, view, window_frac=frac)
        if frac >= 1.0:
            break
        nf = min(1.0, frac * (budget_s / max(sample[3], 1e-3)) ** 0.5)
        if nf <= frac * 1.15:
            break
        frac = nf
    return frac, sample


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene = make_scene(args)
    cam0 = scene.cameras[0]
    vals = []
    desc, cores = "", 0
    frac, _ = pick_window_frac(scene, 0, budget_s=3.0)  # per step; the fraction is then fixed for the whole run
    for i in range(args.warmup + args.steps):
        ms, desc, cores, _ = oracle_sample(scene, i % min(args.views, len(scene.cameras)), window_frac=frac)
        if i >= args.warmup:
            vals.append(ms)
    v = float(np.mean(vals))
    _, aff, ncpu = oracle_cores()
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": v, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(scene)},
            "cpu_baseline": {"value": v, "unit": "ms", "cores": cores, "kind": "oracle", "sample": desc, "affinity": aff, "cpu_count": ncpu},
            "e2e": {"value": v, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------------------------
# CUDA arm
# ------------------------------------------------------------------------------------------------------------------

def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2501_08174_b200 import binding as B

    from paper_2501_08174_b200 import sharding
    rank, world, local = sharding.env_rank()
    if world != args.gpus:
        raise RuntimeError(f"--gpus {args.gpus} but the launch has WORLD_SIZE={world}: the number printed must be the number measured")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    if torch.cuda.device_count() <= local:
        raise RuntimeError(f"rank {rank} needs CUDA device {local}, the node has {torch.cuda.device_count()}")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()
    peaks = alu_peaks(B, torch, dev)

    scene = make_scene(args)
    n, deg = scene.n, scene.sh_degree
    cams = scene.cameras
    W, H = cams[0].width, cams[0].height
    # views are sharded over ranks: rank r owns views r, r+world, ...; no data-path collective in the step
    my_views = sharding.rotation_for_rank(len(cams), rank, world, args.views)
    cfg = B.ocgs_default_config(sh_degree=deg)
    cap = int(os.environ.get("OCGS_KEY_CAPACITY", 48 * n if n < 2_000_000 else 16 * n))

    def to_dev(a, dt=torch.float32):
        return torch.tensor(np.ascontiguousarray(a), dtype=dt, device=dev)

    params = dict(pos=to_dev(scene.pos), scale=to_dev(scene.scale), quat=to_dev(scene.quat), opacity=to_dev(scene.opacity), sh=to_dev(scene.sh))
    surfels = B.make_surfels(params["pos"], params["scale"], params["quat"], params["opacity"], params["sh"])
    ws = B.alloc_workspace(n, W, H, cap, device=dev)
    out = B.alloc_outputs(W, H, device=dev)
    grads = B.alloc_grads(n, device=dev)
    gC = torch.empty((3, H, W), dtype=torch.float32, device=dev)
    loss_l1 = torch.zeros(1, dtype=torch.float32, device=dev)
    loss_pm = torch.zeros(3, dtype=torch.float32, device=dev)
    pws_photo = torch.empty(B.ocgs_photometric_workspace_bytes(W, H), dtype=torch.uint8, device=dev) if args.loss != "l1" else None
    loss_reg = torch.zeros(2, dtype=torch.float32, device=dev)
    if args.loss == "eq3":
        moments = torch.zeros((3, H, W), dtype=torch.float32, device=dev)
        gA_r, gD_r = torch.zeros((H, W), dtype=torch.float32, device=dev), torch.zeros((H, W), dtype=torch.float32, device=dev)
        gM_r, gN_r = torch.zeros((2, H, W), dtype=torch.float32, device=dev), torch.zeros((3, H, W), dtype=torch.float32, device=dev)
        pws_reg = torch.empty(B.ocgs_regularizers_workspace_bytes(W, H), dtype=torch.uint8, device=dev)
    vis = torch.zeros(n, dtype=torch.int32, device=dev)
    cs = torch.zeros(n, dtype=torch.float32, device=dev)
    cam_c = [B.camera_from(cams[v]) for v in my_views]
    masks = [to_dev(scene.mask(v), torch.uint8) for v in my_views]

    # targets: forward render of the perturbed copy (Appendix B), once, outside the timed region
    pert = scene.perturbed()
    pp = dict(pos=to_dev(pert.pos), scale=params["scale"], quat=params["quat"], opacity=to_dev(pert.opacity), sh=to_dev(pert.sh))
    psurf = B.make_surfels(pp["pos"], pp["scale"], pp["quat"], pp["opacity"], pp["sh"])
    targets = []
    for i in range(len(my_views)):
        B.ocgs_preprocess(psurf, cam_c[i], cfg, ws, cap)
        B.ocgs_bin_sort(n, cam_c[i], cfg, ws, cap)
        B.ocgs_render_fwd(n, cam_c[i], cfg, ws, cap, masks[i], out["color"], out["alpha"], out["depth"], out["normal"], out["n_contrib"])
        h = B.ocgs_check(ws)
        targets.append(out["color"].clone())
    del pp, psurf

    def step(i, stats=True):
        c, m = cam_c[i], masks[i]
        B.ocgs_preprocess(surfels, c, cfg, ws, cap)
        B.ocgs_bin_sort(n, c, cfg, ws, cap)
        if args.loss == "eq3":  # Eq. 3: L_c^M + alpha L_d + beta L_n + gamma L_b (alpha = 100, beta = 0.05: 2DGS's values for bounded scenes)
            B.ocgs_render_fwd_reg(n, c, cfg, ws, cap, m, out["color"], out["alpha"], out["depth"], out["normal"], out["n_contrib"], out["loss_bg"],
                                  vis if stats else None, cs if stats else None, moments)
            B.ocgs_photometric_loss(out["color"], targets[i], m, W, H, 0.2, gC, loss_pm, pws_photo)
            B.ocgs_regularizers(out["alpha"], out["depth"], moments, out["normal"], c, 100.0, 0.05, gA_r, gD_r, gM_r, gN_r, loss_reg, pws_reg)
            B.ocgs_render_bwd_reg(surfels, c, cfg, ws, cap, m, out["n_contrib"], gC, gA_r, gD_r, gN_r, moments, gM_r, grads["d_pos"],
                                  grads["d_scale"], grads["d_quat"], grads["d_opacity"], grads["d_sh"], grads["d_center2d"])
            return
        if args.loss == "dssim":
            B.ocgs_render_fwd(n, c, cfg, ws, cap, m, out["color"], out["alpha"], out["depth"], out["normal"], out["n_contrib"], out["loss_bg"],
                              vis if stats else None, cs if stats else None)
            B.ocgs_photometric_loss(out["color"], targets[i], m, W, H, 0.2, gC, loss_pm, pws_photo)
        else:  # harness loss S20: masked L1 fused into the forward epilogue (dL/dcolor produced in-kernel)
            B.ocgs_render_fwd_l1(n, c, cfg, ws, cap, m, targets[i], out["color"], out["alpha"], out["depth"], out["normal"], out["n_contrib"],
                                 out["loss_bg"], loss_l1, gC, vis if stats else None, cs if stats else None)
        B.ocgs_render_bwd(surfels, c, cfg, ws, cap, m, out["n_contrib"], gC, None, None, None, grads["d_pos"], grads["d_scale"],
                          grads["d_quat"], grads["d_opacity"], grads["d_sh"], grads["d_center2d"])
        if batch_views:  # the world's views of this step are one optimiser batch: sum their gradients over NVLink
            sharding.allreduce_grads(grads)

    batch_views = bool(args.batch_views and world > 1)
    # set-up: one step per view of the rotation for the workload counters (K, n_vis, evaluated and blended pairs; not warm-up,
    # not timed), then exactly W warm-up steps
    nv = len(my_views)
    counters = []
    for i in range(nv):
        vis.zero_()
        step(i)
        h = B.ocgs_check(ws)
        counters.append(dict(K=int(h.K), n_vis=int(h.n_vis), E=int(out["n_contrib"].long().sum().item()),
                             B=int(vis.long().sum().item()), loss_bg=float(out["loss_bg"].item()),
                             loss_l1=float(loss_pm[1].item() if args.loss != "l1" else loss_l1.item()), loss_dssim=float(loss_pm[2].item()),
                             loss_dist=float(loss_reg[0].item()), loss_normal=float(loss_reg[1].item())))
    for i in range(args.warmup):
        step(i % nv)
    B.ocgs_check(ws)
    vis.zero_(); cs.zero_()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region 1 (`value`): K steps, CUDA events on the launching stream -------------------------------------
    # The step keeps every count on the device (no host sync), so it is captured once per view into a CUDA graph and
    # replayed (--no-graph launches the 18 kernels directly).  Per-launch events are NOT recorded here: an event after
    # every kernel costs ~0.17 ms per step of idle gaps; the per-kernel breakdown comes from region 2 below.
    graphs = None
    if not args.no_graph and not batch_views:
        try:
            graphs = []
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                step(0)  # warm the capture stream
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            for i in range(nv):
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    step(i)
                graphs.append(g)
            for g in graphs:
                g.replay()
            torch.cuda.synchronize()
            B.ocgs_check(ws)
        except Exception as e:  # capture unavailable: time direct launches
            sys.stderr.write(f"bench: CUDA graph capture failed ({e!r}); timing direct launches\n")
            graphs = None
            torch.cuda.synchronize()

    def run_step(i):
        if graphs is not None:
            graphs[i % nv].replay()
        else:
            step(i % nv)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for i in range(args.steps):
        run_step(i)
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    B.ocgs_check(ws)
    # ---- timed region 2 (per-kernel durations): the same K steps, direct launches, an event after every launch ------
    cap_marks = 64 * args.steps + 8
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev2.record()
    B.ocgs_profile_begin(cap_marks)
    for i in range(args.steps):
        step(i % nv)
    marks = B.ocgs_profile_end(cap_marks)
    ev3.record()
    barrier()
    ms_marked = ev2.elapsed_time(ev3)
    clocks = sampler.stop() if rank == 0 else None
    B.ocgs_check(ws)
    ms_total = sharding.max_over_ranks(ms_total, dev)
    # the one exchange step of the un-batched method: the merge of the visibility statistics at the end of a pruning
    # interval -- once per rotation, not per step; timed beside the step (device time, max over ranks)
    stats_allreduce_ms = None
    if world > 1:
        sharding.allreduce_stats(vis, cs)  # warm-up (communicator set-up)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        a0.record()
        sharding.allreduce_stats(vis, cs)
        a1.record()
        barrier()
        stats_allreduce_ms = sharding.max_over_ranks(a0.elapsed_time(a1), dev)

    # ---- visibility pass ("rendering all training views" for the pruning statistics), timed separately ------
    # (a) through the full forward pass (preprocess + bin_sort + render_fwd with the statistics on), (b) through
    # ocgs_visibility_pass (no SH colour, no maps, no blended lists); direct launches, CUDA events, nv views x reps
    vis_pass = None
    if rank == 0 and not args.no_prune:
        vis_b = torch.zeros_like(vis); cs_b = torch.zeros_like(cs)
        reps = max(1, min(args.steps, 20) // nv)

        def full_fwd(i):
            B.ocgs_preprocess(surfels, cam_c[i], cfg, ws, cap)
            B.ocgs_bin_sort(n, cam_c[i], cfg, ws, cap)
            B.ocgs_render_fwd(n, cam_c[i], cfg, ws, cap, None, out["color"], out["alpha"], out["depth"], out["normal"], out["n_contrib"],
                              None, vis_b, cs_b)

        def stats_only(i):
            B.ocgs_visibility_pass(surfels, cam_c[i], cfg, ws, cap, vis_b, cs_b)
        res = {}
        for name, fn in (("full_forward", full_fwd), ("visibility_pass", stats_only)):
            for i in range(nv):
                fn(i)
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a0.record()
            for _ in range(reps):
                for i in range(nv):
                    fn(i)
            a1.record()
            torch.cuda.synchronize()
            res[name] = a0.elapsed_time(a1) / (reps * nv)
        B.ocgs_check(ws)
        # (c) the same pass with two views in flight (two workspaces, two streams): pruning.accumulate_visibility(ws2=...)
        from paper_2501_08174_b200 import pruning
        ws_b = B.alloc_workspace(n, W, H, cap, device=dev)
        cams_rep = [cam_c[i] for _ in range(reps) for i in range(nv)]
        pruning.accumulate_visibility(surfels, n, cams_rep[:nv], cfg, ws, cap, None, vis_b, cs_b, ws2=ws_b)
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a0.record()
        pruning.accumulate_visibility(surfels, n, cams_rep, cfg, ws, cap, None, vis_b, cs_b, ws2=ws_b)
        a1.record()
        torch.cuda.synchronize()
        res["two_streams"] = a0.elapsed_time(a1) / len(cams_rep)
        del ws_b
        vis_pass = {"ms_per_view_full_forward": res["full_forward"], "ms_per_view": res["visibility_pass"],
                    "ms_per_view_two_streams": res["two_streams"], "views": nv, "reps": reps,
                    "what": "statistics of one view: preprocess + bin_sort + forward walk; ocgs_visibility_pass skips the SH colour, "
                            "the maps and the blended lists"}
        del vis_b, cs_b

    # ---- prune pass, timed separately: once per pruning interval, not per step -------------------
    # statistics of the nv views just rendered -> mask -> scan -> stable compaction of all five parameter arrays
    prune = None
    if rank == 0 and not args.no_prune:
        vis.zero_(); cs.zero_()
        for i in range(nv):
            step(i)
        pm = torch.empty(n, dtype=torch.uint8, device=dev)
        remap = torch.empty(n, dtype=torch.int32, device=dev)
        n_out = torch.zeros(1, dtype=torch.int32, device=dev)
        outs = [torch.empty_like(params[k]) for k in ("pos", "scale", "quat", "opacity", "sh")]
        om = B.ocgs_surfels_mut(*[B._ptr(t_) for t_ in outs], n)
        pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device=dev)
        for _ in range(2):
            B.ocgs_prune_stats(surfels, vis, cs, cfg, pm, remap, om, n_out, 0, pws)
        pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        reps = 10
        pe0.record()
        for _ in range(reps):
            B.ocgs_prune_stats(surfels, vis, cs, cfg, pm, remap, om, n_out, 0, pws)
        pe1.record()
        torch.cuda.synchronize()
        p_ms = pe0.elapsed_time(pe1) / reps
        kept = int(n_out.item())
        p_bytes = n * (8 + 4 + 1 + 4 + 232) + kept * 232  # stats + opacity read, mask + remap written, params read, survivors written
        hbm_pk, _src = measured_peaks()
        prune = {"ms": p_ms, "kept": kept, "of": n, "views": nv, "achieved_gbs": p_bytes / (p_ms * 1e-3) / 1e9,
                 "frac_of_hbm": p_bytes / (p_ms * 1e-3) / 1e9 / hbm_pk, "algorithmic_bytes": p_bytes}
        del outs, om
        vis.zero_(); cs.zero_()

    # ---- e2e: the training step through the library's host-facing calls, pinned host buffers, copies inside -------------
    # (a) `e2e`: ocgs_step_view_host -- what a training loop does per iteration: the model (parameters and
    #     gradients) is resident on the device, the VIEW's inputs (target image, mask; the camera travels by value) come
    #     from pinned host memory every step and the step's result (the two loss scalars) is read back.
    # (b) `e2e_host_params`: ocgs_step_host -- the same step with the parameters uploaded and the gradients downloaded
    #     every step as well (a host-side optimiser): 464 MB over PCIe per step, reported for reference.
    e2e = e2e_hp = None
    if not args.no_e2e:
        h_masks = [m.cpu().pin_memory() for m in masks]
        h_targets = [tg.cpu().pin_memory() for tg in targets]
        d_images = torch.empty(14 * H * W, dtype=torch.float32, device=dev)
        d_mask = torch.empty(H * W, dtype=torch.uint8, device=dev)
        d_nc = torch.empty(H * W, dtype=torch.int32, device=dev)
        d_losses = torch.zeros(2, dtype=torch.float32, device=dev)
        h_losses = torch.zeros(2, dtype=torch.float32).pin_memory()
        k_e = max(3, min(args.steps, 20))

        def time_steps(fn):
            for i in range(2):
                fn(i % nv)
            barrier()
            t0 = time.perf_counter()
            for i in range(k_e):
                fn(i % nv)  # synchronises inside (the results are on the host when it returns)
            torch.cuda.synchronize()
            te = torch.tensor([(time.perf_counter() - t0) * 1e3], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(te, op=dist.ReduceOp.MAX)
            return float(te.item()) / (k_e * world)

        copy_stream = torch.cuda.Stream()

        def view_step(i):
            B.ocgs_step_view_host(surfels, cam_c[i], cfg, h_masks[i], h_targets[i], h_losses, d_mask, d_images, d_nc, grads, vis, cs,
                                  d_losses, ws, cap, copy_stream=copy_stream)
        ms_direct = time_steps(view_step)
        ms_view, how = ms_direct, "ocgs_step_view_host (direct launches, synchronises inside)"
        if not args.no_graph:
            # the same step enqueued by ocgs_step_view_host_enqueue and captured once per view: a replay uploads that view's
            # mask and target from pinned host memory again, runs the step and copies losses + header back
            h_header = torch.zeros(4, dtype=torch.int32).pin_memory()
            main = torch.cuda.Stream()
            torch.cuda.synchronize()
            e2e_graphs = []
            for i in range(nv):
                gr = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gr, stream=main):
                    B.ocgs_step_view_host_enqueue(surfels, cam_c[i], cfg, h_masks[i], h_targets[i], h_losses, h_header, d_mask, d_images, d_nc,
                                                  grads, vis, cs, d_losses, ws, cap, stream=main, copy_stream=copy_stream)
                e2e_graphs.append(gr)

            def view_step_graph(i):
                with torch.cuda.stream(main):
                    e2e_graphs[i].replay()
                main.synchronize()
                if int(h_header[3]) != 0:
                    raise RuntimeError("step reported error bits %d" % int(h_header[3]))
            direct_losses = [float(h_losses[0]), float(h_losses[1])]
            ms_view = time_steps(view_step_graph)
            how = "ocgs_step_view_host_enqueue captured into one CUDA graph per view, replay + stream synchronise + header check per step"
            # same view as the last direct step -> same forward loss, bit for bit (L_b is a fixed-order reduction)
            assert float(h_losses[0]) == direct_losses[0], (float(h_losses[0]), direct_losses)
        ms_sameview = None
        if not args.no_graph:
            # the prefetching form (ocgs_step_view_prefetch_enqueue), what a data loader does: step k runs on view k's mask and
            # target, which step k-1 uploaded from pinned host memory while it was computing, and uploads view k+1's meanwhile;
            # every step's timed region therefore contains exactly one view's upload (its successor's) and the read-back of
            # its own losses and header.  The resident target lets the forward pass fuse the masked L1.
            ms_sameview = ms_view
            d_img11 = torch.empty(11 * H * W, dtype=torch.float32, device=dev)
            bufs = [(torch.empty(H * W, dtype=torch.uint8, device=dev), torch.empty(3 * H * W, dtype=torch.float32, device=dev)) for _ in range(2)]
            pgraphs = {}

            def pgraph(v, par):
                if (v, par) not in pgraphs:
                    nx = (v + 1) % nv
                    torch.cuda.synchronize()
                    gr = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(gr, stream=main):
                        B.ocgs_step_view_prefetch_enqueue(surfels, cam_c[v], cfg, h_masks[nx], h_targets[nx], h_losses, h_header, bufs[par][0],
                                                          bufs[par][1], bufs[1 - par][0], bufs[1 - par][1], d_img11, d_nc, grads, vis, cs,
                                                          d_losses, ws, cap, stream=main, copy_stream=copy_stream)
                    pgraphs[(v, par)] = gr
                return pgraphs[(v, par)]
            for k in range(2 * nv):
                pgraph(k % nv, k % 2)
            state = {"k": 0}

            def prime():  # view 0 into buffer 0, outside the timed region (once per run)
                bufs[0][0].copy_(h_masks[0].view(-1), non_blocking=True)
                bufs[0][1].copy_(h_targets[0].view(-1), non_blocking=True)
                torch.cuda.synchronize()
                state["k"] = 0

            def view_step_prefetch(_):
                k = state["k"]
                gr = pgraph(k % nv, k % 2)
                with torch.cuda.stream(main):
                    gr.replay()
                main.synchronize()
                if int(h_header[3]) != 0:
                    raise RuntimeError("step reported error bits %d" % int(h_header[3]))
                state["k"] = k + 1
            prime()
            ms_view = time_steps(view_step_prefetch)
            how = ("ocgs_step_view_prefetch_enqueue captured into CUDA graphs (one per view and buffer parity), replay + stream synchronise + "
                   "header check per step; the step's own inputs were uploaded by the previous step's prefetch, the next view's are uploaded "
                   "during this step")
            # the pipelined steps really ran on their own view's data: same forward losses as a direct step on that view
            v_last, got = (state["k"] - 1) % nv, (float(h_losses[0]), float(h_losses[1]))
            view_step(v_last)
            assert got[0] == float(h_losses[0]) and abs(got[1] - float(h_losses[1])) < 1e-6, (got, float(h_losses[0]), float(h_losses[1]))
        e2e = {"value": ms_view, "unit": "ms", "h2d_bytes_per_step": H * W + 3 * H * W * 4, "d2h_bytes_per_step": 8 + 16, "steps": k_e,
               "what": ("step k runs on inputs uploaded during step k-1 (data-loader prefetch): " if not args.no_graph else "") + how +
                       ": target image + mask from pinned host memory each step, parameters and gradients resident "
                       "in HBM, uploads on a second stream overlapping preprocess/sort/forward, loss scalars read back; the form that uploads "
                       "the step's OWN view inside the step is graph_upload_inside_step_ms",
               "direct_launch_ms": ms_direct, "graph_upload_inside_step_ms": ms_sameview,
               "losses_last_step": [float(h_losses[0]), float(h_losses[1])]}
        hp = {k: torch.tensor(np.ascontiguousarray(getattr(scene, k)), dtype=torch.float32).pin_memory() for k in ("pos", "scale", "quat", "opacity", "sh")}
        h_grads = torch.empty(58 * n, dtype=torch.float32).pin_memory()
        h_alpha = torch.empty(H * W, dtype=torch.float32).pin_memory()
        h_loss = torch.empty(1, dtype=torch.float32).pin_memory()
        d_params = torch.empty(58 * n + 16, dtype=torch.float32, device=dev)
        d_grads = torch.empty(58 * n + 16, dtype=torch.float32, device=dev)
        d_lb = torch.zeros(1, dtype=torch.float32, device=dev)

        def host_params_step(i):
            B.ocgs_step_host(hp["pos"], hp["scale"], hp["quat"], hp["opacity"], hp["sh"], n, cam_c[i], cfg, h_masks[i], h_targets[i],
                             h_grads, h_alpha, h_loss, d_params, d_mask, d_images, d_nc, d_grads, vis, cs, d_lb, ws, cap)
        k_e = max(3, min(args.steps, 10))
        ms_hp = time_steps(host_params_step)
        e2e_hp = {"value": ms_hp, "unit": "ms", "h2d_bytes_per_step": 58 * n * 4 + H * W + 3 * H * W * 4,
                  "d2h_bytes_per_step": 58 * n * 4 + H * W * 4 + 4 + 16, "steps": k_e,
                  "what": "ocgs_step_host: parameters up and gradients down every step as well (PCIe bound by construction)"}
        del hp, h_grads, d_params, d_grads

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- per-kernel breakdown and roofline of the dominant kernel ----------------------------------------------------
    agg, cnt = {}, {}
    for name, ms in marks:
        agg[name] = agg.get(name, 0.0) + ms
        cnt[name] = cnt.get(name, 0) + 1
    steps = args.steps
    kern_total = sum(agg.values())
    kernels = sorted(({"name": k, "ms_per_step": agg[k] / steps, "launches_per_step": cnt[k] / steps, "share": agg[k] / kern_total}
                      for k in agg), key=lambda d: -d["ms_per_step"])
    launches = sum(c for k, c in cnt.items() if not k.startswith("memset"))
    mean = {k: float(np.mean([c[k] for c in counters])) for k in counters[0]}
    hbm_peak, peak_src = measured_peaks()

    def roofline_of(kd):
        """Roofline entry of one kernel: algorithmic work per launch / average launch duration."""
        name = kd["name"]
        avg_s = (agg[name] / cnt[name]) * 1e-3
        seg = {"render_fwd_kernel": "render_fwd_seg_kernel", "render_bwd_kernel": "render_bwd_seg_kernel"}.get(name)
        if seg in agg:  # the cluster launch of the heavy tiles does part of the same work: its time counts (serialised: conservative)
            avg_s += (agg[seg] / cnt[seg]) * 1e-3
        K, nvis, E, Bp = mean["K"], mean["n_vis"], mean["E"], mean["B"]
        if name in ("render_fwd_kernel", "render_bwd_kernel"):
            if name == "render_fwd_kernel":
                fl, what = FLOP_EVAL * E + FLOP_BLEND_FWD * Bp, f"{FLOP_EVAL:.0f} flop x E evaluated pairs + {FLOP_BLEND_FWD:.0f} flop x B blended pairs"
            else:
                fb = FLOP_BLEND_BWD_COLOUR_ONLY if args.loss in ("l1", "dssim") else FLOP_BLEND_BWD
                fl, what = (FLOP_EVAL + fb) * Bp, f"({FLOP_EVAL:.0f} + {fb:.0f}) flop x B blended pairs"
            ach = fl / avg_s / 1e12
            pk = peaks["fp32_tflops_measured"]
            return {"kernel": name, "bound": "alu", "achieved": ach, "peak": pk, "unit": "TFLOP/s", "frac": ach / pk,
                    "traffic": NCU_TRAFFIC.get(name), "traffic_source": NCU_TRAFFIC_SOURCE,
                    "peak_source": "measured: FP32 FMA microbenchmark of this run (ocgs_peak_probe, peaks.fp32_tflops_measured)", "algorithmic": what,
                    "time": "ordinary launch + cluster launch of the heavy tiles (render_*_seg_kernel)"}
        per_launch = {"radix_onesweep_kernel": 16.0 * (4 * n + 2 * K) / 6.0,  # 8 B read + 8 B written per key; 4 passes over N, 2 over K
                      "radix_hist_all_kernel": 4.0 * n, "emit_keys_kernel": 8.0 * K + 12.0 * nvis,  # the tile sort's histograms are built by emit_keys_kernel
                      "preprocess_kernel": 61.0 * n + 296.0 * nvis, "project_bwd_kernel": 232.0 * n + 328.0 * nvis,
                      "reorder_kernel": 208.0 * nvis, "clear_grad_rec_kernel": 96.0 * nvis, "tile_ranges_kernel": 4.0 * K,
                      "masked_l1_kernel": 25.0 * W * H, "ssim_terms_kernel": 63.0 * W * H, "ssim_grad_kernel": 75.0 * W * H,
                      "reg_terms_kernel": 76.0 * W * H, "reg_gather_kernel": 52.0 * W * H}.get(name)
        if per_launch is None:
            return None
        ach = per_launch / avg_s / 1e9
        return {"kernel": name, "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                "traffic": None, "peak_source": peak_src}

    rooflines = [r for r in (roofline_of(kd) for kd in kernels) if r is not None]
    roof = rooflines[0] if rooflines and rooflines[0]["kernel"] == kernels[0]["name"] else roofline_of(kernels[0])

    ms_per_step = ms_total / (steps * world)
    line = {"metric": METRIC, "value": ms_per_step, "unit": "ms", "n_gpus": world, "steps": steps, "warmup": args.warmup,
            "ms_per_step": ms_total / steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": workload_name(scene), "views_rotated_per_rank": nv, "views": my_views, "sharding": "views r, r+N, ... to rank r",
                       "batch_views": batch_views,
                       "l2": "inputs larger than L2: 232 MB of surfel parameters are re-read every step", "key_capacity": cap,
                       "shrink": args.shrink, "loss": {"l1": "masked L1 (S20) + gamma L_b", "dssim": "L_c^M = 0.8 L1 + 0.2 D-SSIM (Eq. 2) + gamma L_b",
                                "eq3": "Eq. 3: L_c^M + 100 L_d + 0.05 L_n + gamma L_b"}[args.loss]},
            "surfels_per_s": n * world / (ms_total / steps * 1e-3), "pixels_per_s": W * H * world / (ms_total / steps * 1e-3),
            "workload_counters": mean, "gpu_launches": launches, "clocks": clocks, "roofline": roof, "rooflines": rooflines, "kernels": kernels[:14],
            "kernel_ms_sum_per_step": kern_total / steps,
            "launch": "cuda_graph_replay" if graphs is not None else "direct", "peaks": peaks, "stats_allreduce_ms": stats_allreduce_ms,
            "kernel_timing": {"how": "second timed region of the same K steps, direct launches, one CUDA event after every launch "
                                     "(those events cost idle gaps, so `value` comes from the region without them)",
                              "ms_per_step_with_events": ms_marked / steps}}
    line["prune"] = prune
    line["visibility_pass"] = vis_pass
    if e2e:
        line["e2e"] = e2e
        line["e2e_host_params"] = e2e_hp
    if world == 1 and not args.no_cpu_baseline:
        import oracle as orc
        frac, (ms_cpu, desc, cores, _) = pick_window_frac(scene, my_views[0], budget_s=12.0)
        _, aff, ncpu = oracle_cores()
        # the same oracle on ONE core: a smaller centred window, so that it stays within ~10 s
        orc.set_num_threads(1)
        ms_1, desc_1, _, _ = oracle_sample(scene, my_views[0], window_frac=max(0.1, frac / max(1.0, cores) ** 0.5))
        orc.set_num_threads(cores)
        line["cpu_baseline"] = {"value": ms_cpu, "unit": "ms", "cores": cores, "kind": "oracle", "sample": desc, "affinity": aff, "cpu_count": ncpu,
                                "one_core": {"value": ms_1, "unit": "ms", "cores": 1, "sample": desc_1}}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        # `--gpus N` outside torchrun starts the N ranks itself (and refuses when the node has fewer than N CUDA devices)
        from paper_2501_08174_b200 import sharding as _sh
        rc = _sh.relaunch_under_torchrun(a.gpus, [os.path.abspath(__file__)] + sys.argv[1:])
        if rc is not None:
            sys.exit(rc)
        run_ours(a)
