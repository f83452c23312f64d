#!/usr/bin/env python
"""bench.py -- throughput of the BLINK hot path on synthetic workloads, one JSON line (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload station|mwa1|mwa2|sweep256|...]
    python bench.py --impl reference ...        # times the CPU oracle instead (reference arm)

A "step" is one pass of the whole hot path (steps a0-a5 of SURVEY.md section 8: grid every snapshot,
weight, inverse DFT, shift, normalise, real part) over one batch of synthetic visibilities already
resident in HBM, through the public call blink_grid_image (`--path separate`: blink_grid +
blink_image with the uv grids in HBM).  Headline workload = BASELINE.json configs[1] (SKA-Low
station, 100 t x 32 ch x 32640 bl, 256^2); at N = 1 the same process also times configs[2] (MWA
Phase I, 1024^2), configs[3] (MWA Phase II, 4096^2) and the whole configs[4] sweep (128^2 .. 1024^2),
reports them under "workloads", and ends the line with a compact "summary" of every workload's
[ms per step, fraction of the HBM roofline] so that a truncated log still carries them.
"""
from __future__ import annotations

import argparse
import glob
import json
import math
import os
import re
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2405_13478_b200 import shard, synth  # noqa: E402


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
    """SURVEY.md section 8(d), per snapshot: blink_grid reads 8 n_bl and writes 8 N^2; blink_image reads
    8 N^2 and writes 4 N^2; the one-call route has no uv grid in HBM: B_fused = 8 n_bl + 4 N^2
    (count/index tables are per-plan, excluded)."""
    nn = w.n_pix * w.n_pix
    return dict(grid=8 * w.n_bl + 8 * nn, image=12 * nn, sep=8 * w.n_bl + 20 * nn, fused=8 * w.n_bl + 4 * nn)


def image_call_bytes(w, plan, blink):
    """blink_image on the two-call path: what the call has to move is the 4 N^2 image plus the uv cells it
    reads -- the routes read the plan's bounding box (line kernels) or only its occupied cells (residue-class
    kernels), never the whole 8 N^2 grid; crediting 12 N^2 would put the call above the HBM peak."""
    nn = w.n_pix * w.n_pix
    if plan.query_i32(blink.Q_WARP_KERNEL) in (2, 3):
        cells = float(np.mean([plan.n_occ(c) for c in range(w.n_ch)]))
    else:
        cells = float(np.mean([(2 * plan.bbox(c)[0] + 1) * (2 * plan.bbox(c)[1] + 1) for c in range(w.n_ch)]))
    return 4 * nn + 8 * min(nn, cells)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


_UNIT = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}


def kernel_sources_sha16():
    """hash of the kernel sources (csrc/*), written into every ncu summary at capture time and compared here:
    a summary taken before a kernel change says so in the line (`traffic_source.stale`)"""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2405_13478_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload: str, path: str, n_snap: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per STEP of the kernels behind the call, from the newest
    round's committed `ncu --set full` summaries profiles/rNN_<workload>_<path>_fullsize[_<kernel>]_summary.txt
    (written by `python -m paper_2405_13478_b200.ncu_summary`): one file per kernel of the step; a file whose
    capture covered fewer snapshots than the step (one launch pair of the chunked route) carries a
    `# snapshots_in_launch K` line and is scaled by n_snap / K.  None when there is none.  File names, times
    and whether the kernel sources changed since the capture go into the line."""
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_{workload}_{path}_fullsize*_summary.txt")))
    if not files:
        return None, None
    rnd = os.path.basename(files[-1]).split("_")[0]
    files = [f for f in files if os.path.basename(f).startswith(rnd + "_")]
    tot, src, sha = 0.0, [], kernel_sources_sha16()
    for f in files:
        txt = open(f).read()
        scale = 1.0
        m = re.search(r"^# snapshots_in_launch\s+(\d+)", txt, re.M)
        if m:
            scale = n_snap / float(m.group(1))
        for key in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            m = re.search(rf"^{re.escape(key)}\s+([0-9.,]+)\s+(\w+)", txt, re.M)
            if not m or m.group(2) not in _UNIT:
                return None, None
            tot += scale * float(m.group(1).replace(",", "")) * _UNIT[m.group(2)]
        m = re.search(r"^# kernel_sources_sha16\s+(\w+)", txt, re.M)
        src.append({"file": os.path.relpath(f, ROOT), "scaled_by": scale,
                    "stale": (m.group(1) != sha) if m else "unknown (no source hash in the file)"})
    return int(tot), src


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


def workload_config(w, name):
    return {"workload": f"{name}: {w.n_ant} antennas, {w.n_bl} baselines, {w.n_t} time steps x "
                        f"{w.n_ch} channels = {w.n_snapshots} snapshots, {w.n_pix}x{w.n_pix} image, "
                        f"{'natural' if w.weighting == 0 else 'uniform'} weighting",
            "n_ant": w.n_ant, "n_bl": w.n_bl, "n_t": w.n_t, "n_ch": w.n_ch, "n_pix": w.n_pix,
            "weighting": "natural" if w.weighting == 0 else "uniform",
            "l2_policy": "inputs larger than L2: each step streams the whole batch of visibilities and images "
                         "(>= 0.8 GB) through the 126 MB L2"}


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


def cpu_baseline(w, args):
    """The oracle as it stands, timed on this box's host cores, on a bounded sample: (i) all cores
    (OpenMP over snapshots); (ii) ONE thread -- the paper's CPU imager is single-threaded
     -- with gridding and the transform timed separately like its Tables 5-6
    (PAPER.md:493-506, :546-565)."""
    from oracle import oracle as orc
    orc.build()
    n_t_s = ref_time_steps(args, w)
    vis = w.vis(0, n_t_s)
    sel = np.arange(n_t_s * w.n_ch, dtype=np.int64)
    t0 = time.perf_counter()
    out = orc.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel,
                          want_grids=False, want_images=True, n_threads=0)
    dt = time.perf_counter() - t0
    cores = out["threads"]
    # single thread on 1/cores of that sample (same CPU seconds), at least 4 snapshots
    sel1 = sel[:max(min(4, len(sel)), len(sel) // max(cores, 1))]
    t0 = time.perf_counter()
    orc.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel1,
                    want_grids=True, want_images=False, n_threads=1)          # cell rule + gridding only
    dt_grid = time.perf_counter() - t0
    t0 = time.perf_counter()
    orc.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel1,
                    want_grids=False, want_images=True, n_threads=1)          # whole chain
    dt_all = time.perf_counter() - t0
    return {"value": len(sel) / dt, "unit": "images/s", "cores": cores, "kind": "oracle",
            "seconds": dt,
            "sample": f"first {n_t_s} of {w.n_t} time steps x {w.n_ch} channels = {len(sel)} snapshots, "
                      "fp64 gridding + naive separable DFT (O(N^3)), OpenMP over snapshots",
            "single_thread": {"value": len(sel1) / dt_all, "unit": "images/s", "cores": 1,
                              "snapshots": int(len(sel1)), "ms_per_image": 1e3 * dt_all / len(sel1),
                              "gridding_ms_per_image": 1e3 * dt_grid / len(sel1),
                              "dft_ms_per_image": 1e3 * max(dt_all - dt_grid, 0.0) / len(sel1),
                              "note": "gridding = uv cells + accumulate (fp64); dft = weighting + naive separable "
                                      "DFT; the paper's single-threaded CPU imager (FFTW) took 4.6-195 ms gridding "
                                      "and 0.34-1481 ms FFT per image (PAPER.md Table 6, other hardware)"}}


def probe_alu_peak(torch, blink, stream):
    """the fp32 peak is measured in-run, by timing blink_probe_fp32 (a register-only
    kernel, eight independent chains per thread) for scalar / packed adds and FMAs."""
    out = torch.empty(148 * 16 * 256, dtype=torch.float32, device="cuda")
    res = {}
    for op, name in enumerate(["fadd", "ffma", "fadd2", "ffma2"]):
        blink.probe_fp32(op, 64, out)                                  # warm-up
        best = 0.0
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            flops = blink.probe_fp32(op, 2048, out)
            e1.record(stream)
            torch.cuda.synchronize()
            best = max(best, flops / (e0.elapsed_time(e1) / 1e3) / 1e12)
        res[f"{name}_tflops"] = best
    res["how"] = ("blink_probe_fp32 (csrc/blink_probe.cu): 2368 CTAs x 256 threads x 2048 x 64 instructions of one "
                  "kind in 8 independent chains, CUDA events, best of 3; an FMA counts 2 flops, packed f32x2 "
                  "instructions count both lanes")
    return res


def algorithmic_flops(w, plan, blink):
    """fp32 work per snapshot that the method needs (ALU side bound of SURVEY.md section 8(d)):
    gridding 2 adds per kept visibility (Hermitian half-plane), plus the Hermitian two-pass transform,
    a 1-D transform of length N counted 5 N log2 N.  Pass A: kx_max + 1 columns; on the
    warp-per-transform route (wide sparse half-planes) it is what that route computes -- per occupied
    half-plane cell one complex multiply-add into each of 32 partial sums (8 x 32 flops), per column a
    32-point butterfly on each of 32 lanes plus its twiddles.  Pass B: N/2 complex row transforms (two
    real rows each)."""
    n = w.n_pix
    kxm = max(plan.bbox(c)[0] for c in range(w.n_ch))
    fft = 5.0 * n * math.log2(n)
    grid = 2.0 * w.n_bl
    pass_b = (n / 2) * fft
    if plan.query_i32(blink.Q_FUSED_PATH) == 2 and plan.query_i32(blink.Q_WARP_KERNEL) == 2:
        # residue-class kernel: 64 units per snapshot; per unit every occupied half-plane cell takes one complex
        # multiply-add (8 flops; its unit-modulus factor comes from the special-function unit and is not counted),
        # every one of the 512 tile columns a 16-point butterfly plus the two row-pass operands per row pair
        half_cells = np.mean([plan.n_occ(c) for c in range(w.n_ch)]) / 2.0
        pass_a = 64.0 * (half_cells * 8.0 + 512 * (5.0 * 16 * 4 + 4.0 * 16))
        form = "sparse pass A (residue-class kernel)"
    elif plan.query_i32(blink.Q_FUSED_PATH) == 2:
        half_cells = np.mean([plan.n_occ(c) for c in range(w.n_ch)]) / 2.0
        pass_a = half_cells * 8.0 * 32 + (kxm + 1) * (32 * 5.0 * 32 * 5 + 6.0 * n)
        form = "sparse pass A (warp route)"
    elif plan.query_i32(blink.Q_WARP_KERNEL) == 3:
        # k_cols_res (N = 2048 / 4096): N / 8 units per snapshot; per unit one complex multiply-add per occupied
        # half-plane cell and an 8-point butterfly on each of the 1024 tile columns
        half_cells = np.mean([plan.n_occ(c) for c in range(w.n_ch)]) / 2.0
        pass_a = (n / 8.0) * (half_cells * 8.0 + 1024 * 5.0 * 8 * 3)
        form = "sparse pass A (residue-class column pass)"
    else:
        pass_a = (kxm + 1) * fft
        form = "dense pruned pass A"
    return grid + pass_a + pass_b, form


def time_steps(torch, plan, vis, img, uv, steps, warmup, stream, barrier):
    """W untimed + K timed steps, CUDA events on the launching stream; returns (total ms, per-call ms)."""
    fused = uv is None

    def one(ev=None, k=0):
        if fused:
            plan.grid_image(vis, img)
            if ev:
                ev[3 * k + 1].record(stream)
        else:
            plan.grid(vis, uv)
            if ev:
                ev[3 * k + 1].record(stream)
            plan.image(uv, img)
        if ev:
            ev[3 * k + 2].record(stream)
            ev[3 * k + 3].record(stream)

    for _ in range(max(warmup, 3)):
        one()
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3 * steps + 1)]
    ev[0].record(stream)
    for k in range(steps):
        one(ev, k)
    barrier()
    total_ms = ev[0].elapsed_time(ev[3 * steps])
    grid_ms = float(np.mean([ev[3 * k].elapsed_time(ev[3 * k + 1]) for k in range(steps)]))
    image_ms = float(np.mean([ev[3 * k + 1].elapsed_time(ev[3 * k + 2]) for k in range(steps)]))
    time_steps.per_step = [ev[3 * k].elapsed_time(ev[3 * k + 3]) for k in range(steps)]   # best and median
    return total_ms, grid_ms, image_ms


def spread(per_step):
    return {"best": float(np.min(per_step)), "median": float(np.median(per_step)), "worst": float(np.max(per_step)),
            "n": len(per_step)}


def roofline_of(w, plan, blink, name, path, ms_call, dom_bytes, n_snap, peak, peak_src, alu):
    achieved = dom_bytes * n_snap / (ms_call / 1e3) / 1e9
    traffic, src = ncu_traffic(name, path, n_snap)
    flops, form = algorithmic_flops(w, plan, blink)
    tf = flops * n_snap / (ms_call / 1e3) / 1e12
    t_hbm_us = dom_bytes / (peak * 1e9) * 1e6
    side = None
    if alu:
        t_alu_us = flops / (alu["ffma2_tflops"] * 1e12) * 1e6
        side = {"bound": "alu", "flops_per_snapshot": flops, "flop_model": form, "achieved_tflops": tf,
                "peak_tflops_fma": alu["ffma2_tflops"], "frac_of_fma_peak": tf / alu["ffma2_tflops"],
                "peak_tflops_add_only": alu["fadd2_tflops"], "frac_of_add_only_peak": tf / alu["fadd2_tflops"],
                "alu_us_per_snapshot_at_fma_peak": t_alu_us, "hbm_us_per_snapshot_at_peak": t_hbm_us,
                "binding": "alu" if t_alu_us > t_hbm_us else "hbm"}
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "frac_is": "algorithmic bytes / CUDA-event time / measured copy peak (never the ncu traffic)",
            "traffic": traffic, "traffic_source": src, "peak_source": peak_src,
            "algorithmic_bytes_per_snapshot": dom_bytes, "atomics": "none (atomic-free design)"}, side


def extra_workload(torch, blink, name, steps, stream, peak, peak_src, alu):
    """configs[2] / configs[4]@512 timed in the same process, through blink_grid_image."""
    w = make_workload(name)
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)
    plan.reserve(w.n_t)
    vis = torch.from_numpy(w.vis()).cuda()
    img = torch.empty((w.n_t, w.n_ch, w.n_pix, w.n_pix), dtype=torch.float32, device="cuda")
    total_ms, call_ms, _ = time_steps(torch, plan, vis, img, None, steps, 3, stream, torch.cuda.synchronize)
    n_snap = w.n_snapshots
    ms = total_ms / steps
    ab = algorithmic_bytes(w)
    roof, side = roofline_of(w, plan, blink, name, "fused", call_ms, ab["fused"], n_snap, peak, peak_src, alu)
    out = {"config": workload_config(w, name), "steps": steps, "ms_per_step": ms,
           "ms_per_step_spread": spread(time_steps.per_step),
           "images_per_s": n_snap / (ms / 1e3), "mvis_per_s": n_snap * w.n_bl / (ms / 1e3) / 1e6,
           "route": {1: "shared-memory (k_fused)",
                     0: "two kernels" + (" (column pass k_cols_res)" if plan.query_i32(blink.Q_WARP_KERNEL) == 3 else ""),
                     2: {2: "residue-class kernel, intermediate in shared memory (k_img1024r)",
                         1: "warp-per-transform ring kernel (k_img1024)"}.get(plan.query_i32(blink.Q_WARP_KERNEL), "?")}[
               plan.query_i32(blink.Q_FUSED_PATH)],
           "images_per_s_vs_sep_roofline": (n_snap / (ms / 1e3)) / (peak * 1e9 / ab["sep"]),
           "roofline": roof, "side_bounds": side}
    plan.close()
    del vis, img
    torch.cuda.empty_cache()
    return out


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
    ap.add_argument("--extra-workloads", default="mwa1,mwa2,sweep128,sweep256,sweep512,sweep1024",
                    help="comma list of further workloads timed in the same process at N = 1 ('' = none)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-corrections", action="store_true",
                    help="skip the measurement of the pre-gridding corrections (SURVEY.md 8(f) item f2)")
    ap.add_argument("--no-cufft-ref", action="store_true",
                    help="skip the library reference (blink_grid + torch.fft.ifft2 = cuFFT C2C + shift/real/scale)")
    ap.add_argument("--no-dynspec", action="store_true",
                    help="skip the side measurement of blink_dynspec (SURVEY.md 8(f) item f4)")
    ap.add_argument("--only-step", action="store_true", help="time the step only (profiling runs)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.only_step:
        args.no_cpu_baseline = args.no_e2e = args.no_corrections = args.no_cufft_ref = args.no_dynspec = True
        args.extra_workloads = ""

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
    t_plan = time.perf_counter()
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)
    t_plan = time.perf_counter() - t_plan
    plan.reserve(w.n_t)
    t_refresh = time.perf_counter()
    plan.refresh(w.ant_enu_m)                    # a0 again + every table rebuilt and swapped in (f2: plan refresh)
    t_refresh = time.perf_counter() - t_refresh
    vis = vis_h.cuda(non_blocking=True)
    shape = (w.n_t, w.n_ch, w.n_pix, w.n_pix)
    fused = args.path in ("fused", "auto")       # blink_grid_image is the fast public call
    args.path = "fused" if fused else "separate"
    uv = None if fused else torch.empty(shape, dtype=torch.complex64, device="cuda")
    img = torch.empty(shape, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        shard.barrier()
        torch.cuda.synchronize()

    # ---- timed region: exactly K steps, CUDA events on the launching stream, clocks sampled during it
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    total_ms, grid_ms, image_ms = time_steps(torch, plan, vis, img, uv, args.steps, args.warmup, stream, barrier)
    clocks = sampler.stop() if rank == 0 else None
    step_spread = spread(time_steps.per_step)
    total_ms = shard.max_over_ranks(total_ms, device="cuda")
    ms_per_step = total_ms / args.steps
    n_snap = w.n_snapshots
    value = world * n_snap / (ms_per_step / 1e3)

    def timed(fn, n):
        for _ in range(3):
            fn()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n):
            fn()
        b.record(stream)
        barrier()
        return a.elapsed_time(b) / n

    # ---- f2, pre-gridding corrections: (i) fused into the gridder's load -- the same step
    # with the plan's factor table applied to every visibility as it is read, no extra HBM traffic;
    # (ii) the stand-alone pass blink_correct, 16 bytes per visibility
    corr = None
    if not args.no_corrections:
        rng = np.random.default_rng(w.seed + 7)
        n_ant = w.ant_enu_m.shape[0]
        gains = rng.uniform(0.5, 2.0, (w.n_ch, n_ant)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (w.n_ch, n_ant)))
        plan.set_corrections(gains, rng.uniform(0.0, 300.0, n_ant), 0.1, -0.2)
        vis_c = torch.empty_like(vis)
        c_ms = timed(lambda: plan.correct(vis, vis_c), args.steps)
        del vis_c
        c_bytes = 16 * vis.numel()
        fused_corr = None
        if hasattr(plan, "apply_corrections"):
            plan.apply_corrections(True)
            f_ms = timed(lambda: (plan.grid_image(vis, img) if fused else (plan.grid(vis, uv), plan.image(uv, img))),
                         args.steps)
            plan.apply_corrections(False)
            fused_corr = {"ms_per_step": f_ms, "step_without_ms": ms_per_step,
                          "extra_over_step": f_ms / ms_per_step - 1.0, "extra_hbm_bytes": 0}
        corr = {"fused_at_load": fused_corr,
                "separate_pass": {"call": "blink_correct", "ms": c_ms, "algorithmic_bytes": c_bytes,
                                  "achieved_gbs": c_bytes / (c_ms / 1e3) / 1e9,
                                  "extra_over_step": c_ms / ms_per_step,
                                  "gvis_per_s": vis.numel() / (c_ms / 1e3) / 1e9}}

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
        n_f = max(1, min(args.steps, 5))
        f_ms = timed(cufft_step, n_f)
        ref_img = cufft_step()
        ours = plan.image(uv_c)
        o_ms = timed(lambda: plan.image(uv_c, ours), n_f)
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
        d_ms = timed(lambda: plan.dynspec(img, 0.1, state, dyn_out), args.steps)
        d_bytes = 8 * img.numel() + 8 * state.numel()
        dyn = {"call": "blink_dynspec", "alpha": 0.1, "ms": d_ms, "algorithmic_bytes": d_bytes,
               "achieved_gbs": d_bytes / (d_ms / 1e3) / 1e9, "images_per_s": n_snap / (d_ms / 1e3)}
        del dyn_out, state

    # ---- end to end through the C ABI with HOST buffers: one blink_grid_image_host call per step --
    # pinned host visibilities in, images back to pinned host memory, chunked and overlapped inside the
    # library on three streams; the copies are inside the timed region
    e2e = None
    if not args.no_e2e:
        img_h = torch.empty(shape, dtype=torch.float32).pin_memory()
        if fused:
            plan.reserve_host(0)                 # the plan's own chunk: about 32 MiB each way

            def e2e_step():
                plan.grid_image_host(vis_h, img_h)
        else:
            def e2e_step():
                vis.copy_(vis_h, non_blocking=True)
                plan.grid(vis, uv)
                plan.image(uv, img)
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
        te = shard.max_over_ranks(e0.elapsed_time(e1) / n_e, device="cuda")
        h2d, d2h = int(vis_h.numel() * vis_h.element_size()), int(img_h.numel() * img_h.element_size())
        e2e = {"value": world * n_snap / (te / 1e3), "unit": "images/s", "ms_per_step": te,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "call": "blink_grid_image_host (C ABI, host pointers)" if fused else "torch copies + blink_grid + blink_image",
               "host_link_gbs_each_way": max(h2d, d2h) / (te / 1e3) / 1e9,
               "note": "bound by the host link (PCIe): the step's 8 n_bl + 4 N^2 bytes per snapshot cross it once each way"}
        del img_h

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rank 0: rooflines
    peak, peak_src = measured_peaks()
    alu = probe_alu_peak(torch, blink, stream)
    ab = algorithmic_bytes(w)
    if fused:
        calls = {"blink_grid_image": (grid_ms, ab["fused"])}
        step_bytes = ab["fused"]
    else:
        ib = image_call_bytes(w, plan, blink)
        calls = {"blink_grid": (grid_ms, ab["grid"]), "blink_image": (image_ms, ib)}
        step_bytes = ab["grid"] + ib
    dom = max(calls, key=lambda k: calls[k][0])
    roof, side = roofline_of(w, plan, blink, args.workload, args.path, calls[dom][0], calls[dom][1], n_snap, peak,
                             peak_src, alu)
    roof["kernel"] = dom
    step_gbs = step_bytes * n_snap / (ms_per_step / 1e3) / 1e9
    chunks = -(-n_snap // max(1, plan.query_i32(blink.Q_IMAGE_CHUNK)))
    fp = plan.query_i32(blink.Q_FUSED_PATH)
    if fused:
        launches_per_step = 1 if fp in (1, 2) else 2 * (-(-n_snap // max(1, plan.query_i32(blink.Q_FUSED_CHUNK))))
    else:
        launches_per_step = 1 + (1 if fp == 2 else 2 * chunks)

    out = {
        "metric": "dirty_images_per_s", "value": value, "unit": "images/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step,
        "ms_per_step_spread": step_spread,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "mvis_per_s": value * w.n_bl / 1e6,
        "config": workload_config(w, args.workload),
        "path": args.path, "per_call_ms": {k: v[0] for k, v in calls.items()},
        "images_per_s_vs_sep_roofline": value / world / (peak * 1e9 / ab["sep"]),
        "roofline": roof,
        "roofline_step": {"bound": "hbm", "achieved": step_gbs, "peak": peak, "unit": "GB/s",
                          "frac": step_gbs / peak, "algorithmic_bytes_per_snapshot": step_bytes},
        "side_bounds": side, "alu_peak": alu,
        "plan_create_s": t_plan, "plan_refresh_s": t_refresh,
        "f2_corrections": corr, "cufft_reference": cufft,
        "f4_dynspec": dict(dyn, frac_of_hbm_peak=dyn["achieved_gbs"] / peak) if dyn else None,
        "e2e": e2e, "gpu_launches": launches_per_step * args.steps, "clocks": clocks,
    }
    if corr:
        corr["separate_pass"]["frac_of_hbm_peak"] = corr["separate_pass"]["achieved_gbs"] / peak
    plan.close()
    del vis, img, uv
    torch.cuda.empty_cache()
    # ---- the other workloads north_star names, in the same process (N = 1 only)
    if world == 1 and args.extra_workloads:
        out["workloads"] = {}
        for name in [x for x in args.extra_workloads.split(",") if x and x != args.workload]:
            out["workloads"][name] = extra_workload(torch, blink, name, max(3, min(args.steps, 5)), stream, peak,
                                                    peak_src, alu)
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(w, args)
    # ---- last key, short: every workload's [ms per step, fraction of the HBM roofline on the one-call bytes]
    # (north_star's targets are station and mwa1 >= 0.60; DESIGN.md section 7 says which are met)
    sm = {args.workload: [round(ms_per_step, 4), round(out["roofline_step"]["frac"], 3)]}
    for name, r in out.get("workloads", {}).items():
        sm[name] = [round(r["ms_per_step"], 4), round(r["roofline"]["frac"], 3)]
    out["summary"] = {"ms_per_step,frac_of_hbm_roofline": sm, "path": args.path}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
