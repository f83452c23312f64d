#!/usr/bin/env python
"""bench.py -- throughput of the BLINK hot path (blink_grid + blink_image) on synthetic workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload station|mwa1|mwa2|sweep256|...]
    python bench.py --impl reference ...        # times the CPU oracle instead (reference arm)

A "step" is one pass of the whole hot path (grid every snapshot, image every snapshot) over one
batch of synthetic visibilities already resident in HBM.  Prints ONE JSON line (rank 0).
Default workload = BASELINE.json configs[1] (SKA-Low station, 100 t x 32 ch x 32640 bl, 256^2).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2405_13478_b200 import synth  # noqa: E402


def make_workload(name: str):
    if name == "station":
        return synth.config_station()
    if name == "tiny":
        return synth.config_tiny()
    if name == "mwa1":
        return synth.config_mwa1()
    if name == "mwa2":
        return synth.config_mwa2()
    if name.startswith("sweep"):
        return synth.config_sweep(int(name[5:]))
    raise SystemExit(f"unknown workload {name}")


def algorithmic_bytes(w):
    """per snapshot, blink_grid reads 8 n_bl and writes 8 N^2; blink_image
    reads 8 N^2 and writes 4 N^2 (count/index tables are per-plan, excluded)."""
    nn = w.n_pix * w.n_pix
    return dict(grid=8 * w.n_bl + 8 * nn, image=12 * nn, step=8 * w.n_bl + 20 * nn)


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch at the bench's own
# size, from `ncu --set full` captures (profiles/r01_README.md); None where no capture exists
NCU_TRAFFIC_BYTES = {("station", "fused", 100): 848_063_232 + 784_796_416,      # k_fused<256,512,3,1>
                     ("mwa1", "fused", 100): 175_624_704 + 10_052_818_000}      # k_img1024 (profiles/r01aa_k_img1024_summary.txt)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.proc = gpu_index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
            except ValueError:
                continue
            for nm, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(smax)) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def ref_time_steps(args, w, scale=1.0):
    """Bounded oracle sample: ~10-30 s of host work (naive separable DFT is O(N^3) per snapshot)."""
    if args.ref_time_steps > 0:
        return max(1, min(w.n_t, args.ref_time_steps))
    target = {32: 1 << 20, 64: 1 << 18, 128: 1 << 15, 256: 4096, 512: 512, 1024: 96, 2048: 24, 4096: 24}
    snaps = max(1, int(target.get(w.n_pix, 64) * scale))
    return max(1, min(w.n_t, -(-snaps // w.n_ch)))


def run_reference(args, w):
    """Reference arm = the CPU oracle as it stands, on the host cores, on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    orc.build()
    n_t_s = ref_time_steps(args, w, 0.25)   # per step; K + W steps must end within minutes
    vis = w.vis(0, n_t_s)
    sel = np.arange(n_t_s * w.n_ch, dtype=np.int64)
    per = []
    threads = 1
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        out = orc.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel,
                              want_grids=False, want_images=True, n_threads=0)
        dt = time.perf_counter() - t0
        threads = out["threads"]
        if it >= args.warmup:
            per.append(dt)
    ms = 1e3 * float(np.mean(per))
    val = len(sel) / (ms / 1e3)
    sample = f"{n_t_s} of {w.n_t} time steps x {w.n_ch} channels = {len(sel)} snapshots per step"
    print(json.dumps({
        "impl": "reference", "metric": "dirty_images_per_s", "value": val, "unit": "images/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "mvis_per_s": val * w.n_bl / 1e6,
        "config": workload_config(w, args.workload),
        "cpu_baseline": {"value": val, "unit": "images/s", "cores": threads, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "images/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_config(w, name):
    return {"workload": f"{name}: {w.n_ant} antennas, {w.n_bl} baselines, {w.n_t} time steps x "
                        f"{w.n_ch} channels = {w.n_snapshots} snapshots, {w.n_pix}x{w.n_pix} image, "
                        f"{'natural' if w.weighting == 0 else 'uniform'} weighting",
            "n_ant": w.n_ant, "n_bl": w.n_bl, "n_t": w.n_t, "n_ch": w.n_ch, "n_pix": w.n_pix,
            "weighting": "natural" if w.weighting == 0 else "uniform",
            "l2_policy": "inputs larger than L2: each step streams vis, uv grids and images "
                         "(>= 0.8 GB each) through the 126 MB L2"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="station")
    ap.add_argument("--impl", default="blink", choices=["blink", "reference"])
    ap.add_argument("--n-t", type=int, default=0, help="override time steps per batch (0 = config)")
    ap.add_argument("--ref-time-steps", type=int, default=0,
                    help="time steps per step of the CPU reference / cpu_baseline sample "
                         "(0 = sized for roughly 10-30 s of CPU work)")
    ap.add_argument("--path", default="auto", choices=["auto", "separate", "fused"],
                    help="separate = blink_grid + blink_image (uv grid in HBM); fused = blink_grid_image; "
                         "auto = fused")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-corrections", action="store_true",
                    help="skip the side measurement of blink_correct (SURVEY.md 8(f) item f2)")
    ap.add_argument("--no-cufft-ref", action="store_true",
                    help="skip the library reference (blink_grid + torch.fft.ifft2 = cuFFT C2C + shift/real/scale)")
    ap.add_argument("--no-dynspec", action="store_true",
                    help="skip the side measurement of blink_dynspec (SURVEY.md 8(f) item f4)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    w = make_workload(args.workload)
    if args.n_t > 0:
        w.n_t = args.n_t
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import torch.distributed as dist
    from paper_2405_13478_b200 import blink

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    blink.load()

    # ---- inputs: every rank images its own full batch (independent snapshots, no collective)
    w.seed = w.seed + 1000 * rank if rank else w.seed
    vis_h = torch.from_numpy(w.vis()).pin_memory()
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)
    plan.reserve(w.n_t)
    vis = vis_h.cuda(non_blocking=True)
    shape = (w.n_t, w.n_ch, w.n_pix, w.n_pix)
    fused = args.path in ("fused", "auto")       # blink_grid_image is the fast public call
    args.path = "fused" if fused else "separate"
    uv = None if fused else torch.empty(shape, dtype=torch.complex64, device="cuda")
    img = torch.empty(shape, dtype=torch.float32, device="cuda")
    img_h = torch.empty(shape, dtype=torch.float32).pin_memory()
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        if fused:
            plan.grid_image(vis, img)
        else:
            plan.grid(vis, uv)
            plan.image(uv, img)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()

    # ---- timed region: exactly K steps, CUDA events on the launching stream
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3 * args.steps + 1)]
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    ev[0].record(stream)
    for k in range(args.steps):
        if fused:
            plan.grid_image(vis, img)
            ev[3 * k + 1].record(stream)
        else:
            plan.grid(vis, uv)
            ev[3 * k + 1].record(stream)
            plan.image(uv, img)
        ev[3 * k + 2].record(stream)
        ev[3 * k + 3].record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = ev[0].elapsed_time(ev[3 * args.steps])
    grid_ms = float(np.mean([ev[3 * k].elapsed_time(ev[3 * k + 1]) for k in range(args.steps)]))
    image_ms = float(np.mean([ev[3 * k + 1].elapsed_time(ev[3 * k + 2]) for k in range(args.steps)]))
    t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    n_snap = w.n_snapshots
    value = world * n_snap / (ms_per_step / 1e3)

    # ---- side measurement, outside the step: blink_correct (f2), a streaming complex multiply of the
    # whole batch by the plan's factor table; algorithmic bytes 16 per visibility (read 8, write 8)
    corr = None
    if not args.no_corrections:
        rng = np.random.default_rng(w.seed + 7)
        n_ant = w.ant_enu_m.shape[0]
        gains = rng.uniform(0.5, 2.0, (w.n_ch, n_ant)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (w.n_ch, n_ant)))
        plan.set_corrections(gains, rng.uniform(0.0, 300.0, n_ant), 0.1, -0.2)
        vis_c = torch.empty_like(vis)
        for _ in range(3):
            plan.correct(vis, vis_c)
        barrier()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        for _ in range(args.steps):
            plan.correct(vis, vis_c)
        c1.record(stream)
        barrier()
        c_ms = c0.elapsed_time(c1) / args.steps
        c_bytes = 16 * vis.numel()
        corr = {"call": "blink_correct", "ms": c_ms, "algorithmic_bytes": c_bytes,
                "achieved_gbs": c_bytes / (c_ms / 1e3) / 1e9, "gvis_per_s": vis.numel() / (c_ms / 1e3) / 1e9}
        del vis_c

    # ---- library reference timed beside the hand-written transform (north_star item 3):
    # the paper's own design -- a dense batched C2C inverse FFT (cuFFT through torch.fft.ifft2) on the
    # uv grids of blink_grid, then weighting, fftshift, real part and 1/norm as torch elementwise ops --
    # on a chunk of the batch that keeps the extra buffers under ~2 GB each.  Context, not the product.
    cufft = None
    if not args.no_cufft_ref:
        per_t = w.n_ch * w.n_pix * w.n_pix * 8
        n_tc = int(max(1, min(w.n_t, (2 << 30) // per_t)))
        uv_c = plan.grid(vis[:n_tc].contiguous())
        scale = torch.tensor([1.0 / plan.norm(c) if plan.norm(c) > 0 else 0.0 for c in range(w.n_ch)],
                             dtype=torch.float32, device="cuda").view(1, w.n_ch, 1, 1)
        wgt = None
        if w.weighting == synth.UNIFORM:
            cnt = torch.from_numpy(np.stack([plan.counts(c) for c in range(w.n_ch)]).astype(np.float32)).cuda()
            wgt = torch.where(cnt > 0, 1.0 / cnt.clamp(min=1.0), torch.zeros_like(cnt)).unsqueeze(0)

        def cufft_step():
            g = uv_c if wgt is None else uv_c * wgt
            f = torch.fft.ifft2(g, norm="forward")            # unnormalised inverse, e^{+i...}
            return torch.fft.fftshift(f.real, dim=(-2, -1)) * scale
        for _ in range(3):
            ref_img = cufft_step()
        barrier()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_f = max(1, min(args.steps, 5))
        f0.record(stream)
        for _ in range(n_f):
            ref_img = cufft_step()
        f1.record(stream)
        barrier()
        f_ms = f0.elapsed_time(f1) / n_f
        ours = plan.image(uv_c)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        for _ in range(n_f):
            plan.image(uv_c, ours)
        g1.record(stream)
        barrier()
        o_ms = g0.elapsed_time(g1) / n_f
        peak_img = float(ref_img.abs().max())
        cufft = {"what": "torch.fft.ifft2 (cuFFT C2C inverse, batched) + weighting/fftshift/real/scale as torch ops, "
                         "on blink_grid's uv grids", "snapshots": n_tc * w.n_ch, "ms": f_ms,
                 "images_per_s": n_tc * w.n_ch / (f_ms / 1e3),
                 "blink_image_ms_same_chunk": o_ms, "blink_image_images_per_s": n_tc * w.n_ch / (o_ms / 1e3),
                 "max_abs_diff_vs_blink_image_over_peak": float((ours - ref_img).abs().max()) / peak_img}
        del uv_c, ref_img, ours

    # ---- side measurement, outside the step: blink_dynspec (f4) on the step's own image cube:
    # reference subtraction + transpose to [y][x][ch][t]; algorithmic bytes 8 per voxel
    dyn = None
    if not args.no_dynspec:
        state = torch.zeros((w.n_ch, w.n_pix, w.n_pix), dtype=torch.float32, device="cuda")
        dyn_out = torch.empty((w.n_pix, w.n_pix, w.n_ch, w.n_t), dtype=torch.float32, device="cuda")
        for _ in range(3):
            plan.dynspec(img, 0.1, state, dyn_out)
        barrier()
        d0, d1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        d0.record(stream)
        for _ in range(args.steps):
            plan.dynspec(img, 0.1, state, dyn_out)
        d1.record(stream)
        barrier()
        d_ms = d0.elapsed_time(d1) / args.steps
        d_bytes = 8 * img.numel() + 8 * state.numel()
        dyn = {"call": "blink_dynspec", "alpha": 0.1, "ms": d_ms, "algorithmic_bytes": d_bytes,
               "achieved_gbs": d_bytes / (d_ms / 1e3) / 1e9, "images_per_s": n_snap / (d_ms / 1e3)}
        del dyn_out, state

    # ---- end to end: pinned host visibilities in, images back to pinned host memory, per step
    e2e = None
    if not args.no_e2e:
        from paper_2405_13478_b200.pipeline import HostPipeline
        pipe = HostPipeline(plan, w.n_t) if fused else None

        def e2e_step():
            if pipe is not None:                      # chunked, transfers overlapped with imaging
                pipe.run(vis_h, img_h)
            else:
                vis.copy_(vis_h, non_blocking=True)
                step()
                img_h.copy_(img, non_blocking=True)
        e2e_step()
        barrier()
        n_e = max(1, min(args.steps, 3))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n_e):
            e2e_step()
        e1.record(stream)
        barrier()
        te = torch.tensor([e0.elapsed_time(e1) / n_e], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": world * n_snap / (float(te.item()) / 1e3), "unit": "images/s",
               "ms_per_step": float(te.item()),
               "h2d_bytes_per_step": int(vis_h.numel() * vis_h.element_size()),
               "d2h_bytes_per_step": int(img_h.numel() * img_h.element_size())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline (HBM-bound scan/scatter work), dominant call
    peak, peak_src = measured_peaks()
    ab = algorithmic_bytes(w)
    if fused:
        nn = w.n_pix * w.n_pix
        ab["fused"] = 8 * w.n_bl + 4 * nn          # SURVEY.md 8(d) B_fused: no uv grid in HBM
        calls = {"blink_grid_image": (grid_ms, ab["fused"])}
        ab["step"] = ab["fused"]
    else:
        calls = {"blink_grid": (grid_ms, ab["grid"]), "blink_image": (image_ms, ab["image"])}
    dom = max(calls, key=lambda k: calls[k][0])
    achieved = calls[dom][1] * n_snap / (calls[dom][0] / 1e3) / 1e9
    step_gbs = ab["step"] * n_snap / (ms_per_step / 1e3) / 1e9
    chunks = -(-n_snap // max(1, plan.query_i32(blink.Q_IMAGE_CHUNK)))
    if fused:
        if plan.query_i32(blink.Q_FUSED_PATH) in (1, 2):
            launches_per_step = 1
        else:
            launches_per_step = 2 * (-(-n_snap // max(1, plan.query_i32(blink.Q_FUSED_CHUNK))))
    else:
        launches_per_step = 1 + 2 * chunks
    # side bound: fp32 work of the Hermitian two-pass transform + the gridding adds,
    # against the rate the unit counts give (148 SMs x 128 lanes x SM clock, no FMA); DESIGN.md 7
    import math
    kxm = max(plan.bbox(c)[0] for c in range(w.n_ch))
    flops = 5.0 * w.n_pix * math.log2(w.n_pix) * ((kxm + 1) + w.n_pix / 2) + 4.0 * w.n_bl
    fp32_rate = 148 * 128 * 1.965e9
    t_alu_us, t_hbm_us = flops / fp32_rate * 1e6, ab["step"] / (peak * 1e9) * 1e6
    t_meas_us = ms_per_step * 1e3 / n_snap
    side = {"hbm_us_per_snapshot": t_hbm_us, "alu_us_per_snapshot": t_alu_us,
            "measured_us_per_snapshot": t_meas_us, "binding": "alu" if t_alu_us > t_hbm_us else "hbm",
            "frac_of_binding": max(t_alu_us, t_hbm_us) / t_meas_us,
            "flops_per_snapshot": flops, "fp32_rate_no_fma": fp32_rate}
    roof = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak,
            "traffic": NCU_TRAFFIC_BYTES.get((args.workload, args.path, w.n_t)), "peak_source": peak_src,
            "algorithmic_bytes_per_snapshot": calls[dom][1]}
    roof_hbm = None
    if fused and t_alu_us > t_hbm_us:
        # the one-call path is bound by fp32 arithmetic here (1024^2 and larger): report the ALU roofline
        # of the contract -- flops of the Hermitian two-pass transform + gridding adds per launch over the
        # launch time, against the rate the unit counts give without FMA (butterflies are mostly adds;
        # DESIGN.md section 7) -- and keep the HBM figures beside it
        roof_hbm = roof
        tf = flops * n_snap / (calls[dom][0] / 1e3) / 1e12
        roof = {"bound": "alu", "kernel": dom, "achieved": tf, "peak": fp32_rate / 1e12, "unit": "TFLOP/s",
                "frac": tf / (fp32_rate / 1e12), "traffic": roof_hbm["traffic"],
                "peak_source": "derived: 148 SMs x 128 fp32 lanes x 1.965 GHz, one flop per lane and cycle (DESIGN.md 7)",
                "algorithmic_flops_per_snapshot": flops}
    out = {
        "metric": "dirty_images_per_s", "value": value, "unit": "images/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "mvis_per_s": value * w.n_bl / 1e6,
        "config": workload_config(w, args.workload),
        "path": args.path, "per_call_ms": {k: v[0] for k, v in calls.items()},
        "images_per_s_vs_sep_roofline": value / (peak * 1e9 / (8 * w.n_bl + 20 * w.n_pix * w.n_pix)),
        "roofline": roof, "roofline_hbm": roof_hbm,
        "roofline_step": {"bound": "hbm", "achieved": step_gbs, "peak": peak, "unit": "GB/s",
                          "frac": step_gbs / peak, "algorithmic_bytes_per_snapshot": ab["step"]},
        "side_bounds": side,
        "f2_corrections": dict(corr, frac_of_hbm_peak=corr["achieved_gbs"] / peak) if corr else None,
        "cufft_reference": cufft,
        "f4_dynspec": dict(dyn, frac_of_hbm_peak=dyn["achieved_gbs"] / peak) if dyn else None,
        "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "clocks": clocks,
    }
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(w, args)
    print(json.dumps(out))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def cpu_baseline(w, args):
    """The oracle as it stands, timed on this box's host cores, on a bounded sample."""
    from oracle import oracle as orc
    orc.build()
    n_t_s = ref_time_steps(args, w)
    vis = w.vis(0, n_t_s)
    sel = np.arange(n_t_s * w.n_ch, dtype=np.int64)
    t0 = time.perf_counter()
    out = orc.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel,
                          want_grids=False, want_images=True, n_threads=0)
    dt = time.perf_counter() - t0
    return {"value": len(sel) / dt, "unit": "images/s", "cores": out["threads"], "kind": "oracle",
            "seconds": dt,
            "sample": f"first {n_t_s} of {w.n_t} time steps x {w.n_ch} channels = {len(sel)} snapshots, "
                      "fp64 gridding + naive separable DFT (O(N^3)), OpenMP over snapshots"}


if __name__ == "__main__":
    main()
