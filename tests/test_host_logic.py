"""CPU-only checks of the product's host side: the C-ABI library builds for sm_100a, loads, and
exports every symbol include/blink.h declares; the host table builder produces a gather that
reproduces the oracle's grid; the FFT stage algebra (fft_core.cuh compiled for the host) matches a
naive DFT; and without a GPU the compute entry points fail loudly (no fallback)."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

from paper_2405_13478_b200 import build as blink_build
from paper_2405_13478_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def blink():
    blink_build.build()
    from paper_2405_13478_b200 import blink as b
    b.load()
    return b


def test_library_exports_every_declared_symbol(blink):
    """libblink.so exports exactly the product ABI of include/blink.h and none of the test hooks;
    libblink_testing.so (same sources + BLINK_TESTING_HOOKS) exports both headers' names."""
    lib, tlib = blink.load(), blink.load_testing()
    declared = {}
    for header, names in (("blink.h", blink.EXPORTS), ("blink_testing.h", blink.TESTING_EXPORTS)):
        hdr = open(os.path.join(ROOT, "include", header)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        declared[header] = set(re.findall(r"\b(blink_[a-z0-9_]+)\s*\(", hdr))
        assert declared[header], "no declarations parsed"
        assert declared[header] == set(names)
    for name in declared["blink.h"]:
        assert hasattr(lib, name), f"{name} declared in blink.h but not exported by libblink.so"
        assert hasattr(tlib, name), f"{name} missing from libblink_testing.so"
    for name in declared["blink_testing.h"]:
        assert hasattr(tlib, name), f"{name} declared in blink_testing.h but not exported by libblink_testing.so"
        assert not hasattr(lib, name), f"test hook {name} is in the product library"
    exported = subprocess.run(["nm", "-D", "--defined-only", blink.LIB_PATH], capture_output=True, text=True).stdout
    c_names = {ln.split()[-1] for ln in exported.splitlines() if " T blink_" in ln}
    assert c_names == declared["blink.h"], c_names ^ declared["blink.h"]
    assert lib.blink_version() == 210
    assert ctypes.sizeof(blink.Options) == 64          # blink_options: 8 + 8 int32
    assert lib.blink_strerror(-3).decode().startswith("CUDA")


def test_sass_is_sm100a_with_bulk_copies(blink):
    """The built library carries sm_100a code, and the gridder's band stores are TMA bulk copies
    (SASS UBLKCP), per /opt/skills/guides/B200_PROFILING.md."""
    out = subprocess.run(["cuobjdump", "-sass", blink.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert "UBLKCP" in out


def test_no_gpu_fails_loudly(blink):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lib = blink.load()
    h = ctypes.c_void_p()
    ant = np.zeros((3, 3))
    fr = np.array([1e8])
    rc = lib.blink_plan_create(ctypes.byref(h), ant.ctypes.data, 3, fr.ctypes.data, 1, 32, 2 / 32, 0, None)
    assert rc == blink.ECUDA and not h.value
    assert lib.blink_last_cuda_error().decode() != ""


@pytest.mark.parametrize("cfg", ["tiny", "station", "mwa1"])
def test_host_gather_tables_reproduce_oracle_grid(blink, oracle, cfg):
    w = {"tiny": synth.config_tiny, "station": lambda: synth.config_station(n_t=1, n_ch=1),
         "mwa1": lambda: synth.config_mwa1(n_t=1, n_ch=1)}[cfg]()
    n = w.n_pix
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[0], n, w.pixscale)
    g = blink.host_build_gather(r["cell"], n)
    assert g["n_kept"] == w.n_bl - r["n_dropped"]
    # canonical cells strictly ascending, all in the half-plane ky > 0 or (ky == 0 and kx >= 0)
    cc = g["can_cell"]
    assert np.all(np.diff(cc) > 0)
    iy, ix = cc // n, cc % n
    assert np.all((iy < n // 2) & ((iy > 0) | (ix < n // 2)))
    seg = g["seg_start"]
    assert seg[0] == 0 and seg[-1] == g["n_kept"] and np.all(np.diff(seg) > 0)
    # every kept baseline appears exactly once; ascending baseline order inside each segment
    bl = g["src"] >> 1
    assert np.array_equal(np.sort(bl), np.flatnonzero(r["cell"] >= 0))
    for j in range(g["n_can"]):
        assert np.all(np.diff(bl[seg[j]:seg[j + 1]]) > 0)
    # the gather reproduces the oracle's grid on the canonical half (fp64 arithmetic here)
    vis = w.vis()[0, 0].astype(np.complex128)
    g_ref, _ = oracle.grid(r["cell"], r["cell_conj"], w.vis()[0, 0], n)
    val = np.where(g["src"] & 1, np.conj(vis[bl]), vis[bl])
    sums = np.add.reduceat(val, seg[:-1])
    ref = g_ref.reshape(-1)[cc]
    dc = cc == 0
    assert np.allclose(sums[~dc], ref[~dc], rtol=1e-12, atol=1e-12)
    assert np.allclose(2 * sums[dc].real, ref[dc].real, rtol=1e-12, atol=1e-12)


@pytest.mark.parametrize("cfg,chunk", [("tiny", 62), ("tiny", 496), ("station", 4664), ("station", 32640 // 4)])
def test_fused_gather_tables_on_host(blink, oracle, cfg, chunk):
    """The shared-memory route's phase-S tables (warp-owned cells, chunks, groups of 32 lanes x <= 4
    rows, zero-slot padding), walked on the host the way a warp walks them, give every canonical
    cell's sum -- against numpy's per-segment sums of the same visibilities."""
    w = {"tiny": synth.config_tiny, "station": lambda: synth.config_station(n_t=1, n_ch=1)}[cfg]()
    n = w.n_pix
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[0], n, w.pixscale)
    g = blink.host_build_gather(r["cell"], n)
    vis = w.vis()[0, 0]
    out = blink.host_fused_emulate(r["cell"], n, chunk, vis)
    assert out["n_can"] == g["n_can"]
    bl = g["src"] >> 1
    val = np.where(g["src"] & 1, np.conj(vis[bl]), vis[bl]).astype(np.complex128)
    ref = np.add.reduceat(val, g["seg_start"][:-1])
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(out["sums"] - ref)) <= 1e-5 * scale
    # every baseline is read exactly once: rows x 32 lanes >= kept baselines, groups cover the cells
    assert out["rows"] * 32 >= g["n_kept"] and out["groups"] * 32 >= g["n_can"]


@pytest.mark.parametrize("weighting", ["uniform", "natural"])
def test_residue_route_tables_on_host(blink, oracle, weighting):
    """The residue-class kernel of blink_grid_image at N = 1024 (k_img1024r) walked on the host: its plan
    tables (bins of the occupied half-plane cells dealt to lanes, last-of-bin flags, tile slots, per-column
    bin masks) and its index algebra (y = 64 p + r, 16-point column pass over iy mod 16, operands
    U[y] + i U[y + 512] and the mirrored half, row pair p) reproduce the oracle's image rows of the listed
    residue classes -- on MWA-like cells, dropped baselines and the kx = 0 column included."""
    w = synth.config_mwa1(n_t=1, n_ch=1)
    wt = synth.UNIFORM if weighting == "uniform" else synth.NATURAL
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[0], w.n_pix, w.pixscale)
    assert r["n_dropped"] > 0
    vis = w.vis()
    units = [0, 1, 37, 63]
    out = blink.host_residue_emulate(r["cell"], w.n_pix, wt, vis[0, 0], units)
    assert out["longest_list"] <= 16 and out["positions"] % 32 == 0
    ref = oracle.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, wt, vis, np.array([0], np.int64))["images"][0]
    peak = np.max(np.abs(ref))
    assert len(out["rows"]) == 16 * len(units)
    for y, row in out["rows"].items():
        assert np.max(np.abs(row - ref[y])) <= 2e-6 * peak, f"image row {y}"


@pytest.mark.parametrize("n_pix", [2048, 4096])
def test_residue_column_pass_tables_on_host(blink, oracle, n_pix):
    """k_cols_res (column pass by residue class at N = 2048 / 4096) walked on the host: tables generic in the
    grid size (record and descriptor packing, eight bins per column), columns dealt to the warps by cell
    count with every lane's columns in its own bank, units of eight rows y = (N / 8) y' + r -- against the
    oracle's literal sums on sampled pixels of the unit's rows."""
    w = synth.config_mwa2(n_t=1, n_ch=1)
    if n_pix == 2048:
        w.n_pix, w.pixscale, w.weighting = 2048, 30.0 * synth.ARCSEC, synth.UNIFORM
    n = w.n_pix
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[0], n, w.pixscale)
    vis = w.vis()
    units = [0, n // 8 - 1, 77]
    out = blink.host_residue_emulate(r["cell"], n, w.weighting, vis[0, 0], units)
    assert out["positions"] % 32 == 0 and out["longest_list"] <= 32
    g_ref, cnt = oracle.grid(r["cell"], r["cell_conj"], vis[0, 0], n)
    gw, norm = oracle.weight(g_ref, cnt, w.weighting)
    rng = np.random.default_rng(5)
    ys = np.array(sorted(out["rows"].keys()))
    assert len(ys) == 8 * len(units)
    yx = np.stack([np.repeat(ys, 6), rng.integers(0, n, 6 * len(ys))], axis=1).astype(np.int32)
    px = oracle.dft2_pixels(gw, norm, yx).real
    got = np.array([out["rows"][int(y)][int(x)] for y, x in yx])
    peak = max(np.max(np.abs(px)), abs(oracle.dft2_pixels(gw, norm, np.array([[n // 2, n // 2]], np.int32)).real[0]))
    assert np.max(np.abs(got - px)) <= 5e-6 * peak


def test_fft_stage_algebra_on_host(tmp_path):
    exe = str(tmp_path / "host_fft_check")
    subprocess.run(["g++", "-O1", "-std=c++17", os.path.join(ROOT, "tests", "host_fft_check.cpp"),
                    "-o", exe], check=True)
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0 and out.stdout.strip().endswith("OK"), out.stdout


def test_parallel_for_reports_a_throwing_worker(tmp_path):
    """plan-time host loops (csrc/parallel_for.h): an exception in a worker must come back to the caller,
    not end the process; every index runs once"""
    exe = str(tmp_path / "host_parallel_check")
    subprocess.run(["g++", "-O1", "-std=c++17", "-pthread", os.path.join(ROOT, "tests", "host_parallel_check.cpp"),
                    "-o", exe], check=True)
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0 and out.stdout.strip().endswith("OK"), out.stdout + out.stderr


def test_polyphase_identity_behind_the_large_image_route():
    """The identity k_fused<256, ..., D> rests on (blink_fused.cu): for a grid confined to |k| < N'/2,
    the D N' x D N' image is D x D interleaved N' x N' images of the same cells, each the N' transform
    of the grid times exp(2 pi i (kx a + ky b) / (D N')).  Checked with numpy's FFT on a random
    Hermitian band-limited grid, fftshift and centred pixel coordinates included."""
    rng = np.random.default_rng(12)
    ns, d, reach = 32, 4, 11
    n = ns * d
    g = np.zeros((n, n), np.complex128)           # FFT-native order, DC at [0][0]
    ks = np.arange(-reach, reach + 1)
    for ky in ks:
        for kx in ks:
            g[ky % n, kx % n] = rng.standard_normal() + 1j * rng.standard_normal()
    idx = (-np.arange(n)) % n
    g = g + np.conj(g[idx][:, idx])               # Hermitian
    full = np.fft.fftshift(np.fft.ifft2(g) * n * n).real        # I[Y][X], pixel (n/2, n/2) = phase centre
    got = np.empty_like(full)
    for b in range(d):
        for a in range(d):
            gs = np.zeros((ns, ns), np.complex128)
            for ky in ks:
                for kx in ks:
                    gs[ky % ns, kx % ns] = g[ky % n, kx % n] * np.exp(2j * np.pi * (kx * a + ky * b) / n)
            sub = np.fft.fftshift(np.fft.ifft2(gs) * ns * ns)
            assert np.max(np.abs(sub.imag)) < 1e-9 * np.max(np.abs(sub.real))   # the modulated grid stays Hermitian
            got[b::d, a::d] = sub.real
    assert np.max(np.abs(got - full)) < 1e-10 * np.max(np.abs(full))


def test_bench_reference_arm_runs_on_cpu_and_prints_the_contract_line():
    """`bench.py --impl reference` times the oracle on the host cores and prints ONE JSON line with the
    contract's keys (no GPU involved; rank 0 only under torchrun)."""
    import json
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                          "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-500:]
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "dirty_images_per_s" and d["unit"] == "images/s"
    assert d["value"] > 0 and d["higher_is_better"] is True and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    other = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "tiny",
                            "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=300, env=env)
    assert other.returncode == 0 and other.stdout.strip() == ""      # the other ranks exit 0 without work


def test_bench_traffic_comes_from_summaries_of_the_current_kernels(tmp_path, monkeypatch):
    """bench.py's `roofline.traffic` is read from committed ncu summaries: every workload of the default line
    must resolve to files of the newest round, summed over the kernels of its step (mwa2: two kernels, one
    launch pair scaled to the step), and a summary captured before a kernel change must be flagged -- the
    committed ones must not be: after editing csrc/, re-capture (profiles/r03_README.md has the commands)."""
    import bench
    steps = {"station": 3200, "mwa1": 2400, "mwa2": 480, "sweep128": 4000, "sweep256": 4000, "sweep512": 4000,
             "sweep1024": 4000}
    for name, n_snap in steps.items():
        w = bench.make_workload(name)
        assert w.n_snapshots == n_snap
        traffic, src = bench.ncu_traffic(name, "fused", n_snap)
        assert traffic is not None and src, f"no committed full-size ncu summary for {name}"
        alg = bench.algorithmic_bytes(w)["fused"] * n_snap
        assert 0.9 * alg <= traffic <= 2.0 * alg, (name, traffic, alg)
        for f in src:
            assert f["stale"] is False, f"{f['file']} was captured before the last change under csrc/: re-capture it"
    _, src = bench.ncu_traffic("mwa2", "fused", 480)
    assert len(src) == 2 and all(abs(f["scaled_by"] - 480 / 75) < 1e-12 for f in src)
    # the flag itself: a copy of a summary with another source hash reads as stale, one without a hash as unknown
    prof = tmp_path / "profiles"
    prof.mkdir()
    txt = open(os.path.join(ROOT, src[0]["file"])).read()
    (prof / "r09_x_fused_fullsize_summary.txt").write_text(re.sub(r"(# kernel_sources_sha16) \w+", r"\1 0123456789abcdef", txt))
    (prof / "r09_y_fused_fullsize_summary.txt").write_text(re.sub(r"# kernel_sources_sha16 \w+\n", "", txt))
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "kernel_sources_sha16", lambda: "f" * 16)
    assert bench.ncu_traffic("x", "fused", 75)[1][0]["stale"] is True
    assert str(bench.ncu_traffic("y", "fused", 75)[1][0]["stale"]).startswith("unknown")
    assert bench.ncu_traffic("z", "fused", 75) == (None, None)
