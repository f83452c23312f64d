"""GPU parity at BASELINE.json's FULL sizes, in the launch configurations bench.py times: one
blink_grid_image call over the whole batch (persistent CTAs that image many snapshots each), NaN-
prefilled outputs, every image checked to be written, sampled snapshots against the CPU oracle at
the north_star bar (max|d| <= 1e-4 * image peak).  Plus the sizes the library accepts but the
small-case tests never reach (4096^2 through blink_grid_image, N = 2048)."""
import numpy as np
import pytest

from paper_2405_13478_b200 import synth

pytestmark = pytest.mark.gpu

GRID_TOL = 1e-5
IMG_TOL = 1e-4


def _plan(blink, w, **options):
    return blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, options=options or None)


def _fullsize_grid_image(torch, blink, oracle, w, sel, expect_path, **options):
    vis = w.vis()
    plan = _plan(blink, w, **options)
    assert plan.query_i32(blink.Q_FUSED_PATH) == expect_path
    n_snap = w.n_t * w.n_ch
    img = torch.full((w.n_t, w.n_ch, w.n_pix, w.n_pix), float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(torch.from_numpy(vis).cuda(), img)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(img.view(n_snap, -1).sum(dim=1)).all()), "some image not fully written"
    sel = np.asarray(sel, np.int64)
    ref = oracle.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel)
    imh = img.view(n_snap, w.n_pix, w.n_pix)[torch.from_numpy(sel).cuda()].cpu().numpy()
    for q in range(len(sel)):
        peak = np.max(np.abs(ref["images"][q]))
        err = np.max(np.abs(imh[q] - ref["images"][q]))
        assert err <= IMG_TOL * peak, f"snapshot {sel[q]}: err {err:.3e} peak {peak:.3e}"
    plan.close()


def test_full_size_station_grid_image(torch_cuda, blink, oracle):
    """BASELINE.json configs[1] at FULL size through blink_grid_image -- the kernel instance bench.py's
    headline times (k_fused<256,512,3,1>: 3200 snapshots over 148 persistent CTAs, > 21 snapshots per
    CTA, so the hand-off between snapshots -- region_free, the next snapshot's chunk 0 in the dedicated
    buffer, the clearing of the cell sums -- is what is being tested).  Sampled snapshots include the
    first one of a CTA's second round (148), mid-batch ones and the last."""
    w = synth.config_station()
    n_snap = w.n_t * w.n_ch
    _fullsize_grid_image(torch_cuda, blink, oracle, w, [0, 147, 148, 149, 777, 1600, 3051, n_snap - 1], 1)


def test_full_size_station_grid_image_tensor_cores(torch_cuda, blink, oracle):
    """The same batch through k_fused_tc (tune[7] = 1): > 21 snapshots per CTA with the image of each held in
    TMEM while the next one is gridded."""
    w = synth.config_station()
    n_snap = w.n_t * w.n_ch
    _fullsize_grid_image(torch_cuda, blink, oracle, w, [0, 147, 148, 1600, n_snap - 149, n_snap - 1], 1, tune={7: 1})


@pytest.mark.parametrize("n_pix,sel", [(128, [0, 148, 2222, 3999]), (256, [0, 148, 2222, 3999]),
                                       (1024, [0, 149, 3999])])
def test_full_size_sweep_grid_image(torch_cuda, blink, oracle, n_pix, sel):
    """BASELINE.json configs[4] (1000 t x 4 coarse channels x 32640 bl, dispersed pulse) at 128^2,
    256^2 and 1024^2 (512^2 is in test_gpu_parity.py), full size, one blink_grid_image call: direct
    shared-memory route at 128 / 256, polyphase D = 4 at 1024."""
    w = synth.config_sweep(n_pix)
    _fullsize_grid_image(torch_cuda, blink, oracle, w, sel, 1)


def _sampled_pixel_check(oracle, w, vis, s, im, yx, uv=None):
    """One snapshot of a large image against the oracle on sampled pixels (literal sums over the
    occupied cells), the peak taken at the GPU image's arg-max and cross-checked there."""
    n = w.n_pix
    ch = s % w.n_ch
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[ch], n, w.pixscale)
    g_ref, cnt = oracle.grid(r["cell"], r["cell_conj"], vis[s // w.n_ch, ch], n)
    if uv is not None:
        assert np.max(np.abs(uv - g_ref)) <= GRID_TOL * np.max(np.abs(g_ref))
        assert np.all(uv[g_ref == 0] == 0)
    gw, norm = oracle.weight(g_ref, cnt, w.weighting)
    yp, xp = np.unravel_index(np.argmax(np.abs(im)), im.shape)
    peak = abs(oracle.dft2_pixels(gw, norm, np.array([[yp, xp]], np.int32)).real[0])
    assert abs(peak - abs(im[yp, xp])) <= IMG_TOL * peak
    px = oracle.dft2_pixels(gw, norm, yx).real
    err = np.max(np.abs(im[yx[:, 0], yx[:, 1]] - px))
    assert err <= IMG_TOL * peak, f"snapshot {s}: err {err:.3e} peak {peak:.3e}"


def _pixels(n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    return np.concatenate([rng.integers(0, n, (200, 2)),
                           [[0, 0], [n - 1, n - 1], [n // 2, n // 2], [n // 2 - 1, n // 2 + 1], [0, n - 1],
                            [n // 2, 0], [n - 1, n // 2]]]).astype(np.int32)


def test_mwa2_4096_grid_image_sampled_pixels(torch_cuda, blink, oracle):
    """BASELINE.json configs[3] (4096^2) through blink_grid_image (two-kernel route: column pass by
    residue class straight from the visibilities, k_cols_res<12>, + k_image_rows<4096>), more snapshots
    than one time step so the channel index wraps; every image fully written, every snapshot checked on
    sampled pixels."""
    torch = torch_cuda
    w = synth.config_mwa2(n_t=2, n_ch=3)
    vis = w.vis()
    plan = _plan(blink, w)
    assert plan.query_i32(blink.Q_FUSED_PATH) == 0 and plan.query_i32(blink.Q_WARP_KERNEL) == 3
    n = w.n_pix
    img = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(torch.from_numpy(vis).cuda(), img)
    torch.cuda.synchronize()
    assert torch.isfinite(img).all(), "image not fully written"
    imh = img.cpu().numpy().reshape(-1, n, n)
    yx = _pixels(n, 41)
    for s in range(w.n_t * w.n_ch):
        _sampled_pixel_check(oracle, w, vis, s, imh[s], yx)
    plan.close()


@pytest.mark.parametrize("weighting", [synth.NATURAL, synth.UNIFORM])
def test_n2048_all_calls(torch_cuda, blink, oracle, weighting):
    """N = 2048 (accepted by blink_plan_create, instantiated as k_image_rows<2048> etc.): the MWA
    Phase II layout imaged at 30 arcsec per pixel.  Indices and counts bit-exact, blink_grid at the
    grid bar, blink_image and blink_grid_image on sampled pixels, both weightings."""
    torch = torch_cuda
    w = synth.config_mwa2(n_t=2, n_ch=2)
    w.n_pix, w.pixscale, w.weighting = 2048, 30.0 * synth.ARCSEC, weighting
    vis = w.vis()
    plan = _plan(blink, w)
    assert plan.query_i32(blink.Q_WARP_KERNEL) == 3      # column pass: k_cols_res<11>
    n = w.n_pix
    for ch in range(w.n_ch):
        r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[ch], n, w.pixscale)
        assert np.array_equal(plan.cell_idx(ch), r["cell"])
        assert np.array_equal(plan.counts(ch), oracle.counts(r["cell"], r["cell_conj"], n))
    v = torch.from_numpy(vis).cuda()
    uv = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.complex64, device="cuda")
    plan.grid(v, uv)
    img = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.float32, device="cuda")
    plan.image(uv, img)
    img2 = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(v, img2)
    torch.cuda.synchronize()
    assert torch.isfinite(uv.view(torch.float32)).all() and torch.isfinite(img).all() and torch.isfinite(img2).all()
    uvh = uv.cpu().numpy().reshape(-1, n, n)
    imh, imh2 = img.cpu().numpy().reshape(-1, n, n), img2.cpu().numpy().reshape(-1, n, n)
    yx = _pixels(n, 43)
    for s in range(w.n_t * w.n_ch):
        _sampled_pixel_check(oracle, w, vis, s, imh[s], yx, uv=uvh[s])
        _sampled_pixel_check(oracle, w, vis, s, imh2[s], yx)
    plan.close()


@pytest.mark.parametrize("n_pix", [2048, 4096])
def test_residue_column_pass_matches_line_kernels(torch_cuda, blink, n_pix):
    """k_cols_res (column pass by residue class: cells of a snapshot in shared memory, units of 8 image rows,
    rows leaving as bulk copies, CTAs that change snapshot and channel mid-run) against the line kernels
    k_cols_from_vis / k_image_cols (option warp_route = -1) on EVERY pixel of every snapshot, for
    blink_grid_image and for blink_image on blink_grid's uv grids; bit-identical from call to call."""
    torch = torch_cuda
    w = synth.config_mwa2(n_t=3, n_ch=2)
    if n_pix == 2048:
        w.n_pix, w.pixscale, w.weighting = 2048, 30.0 * synth.ARCSEC, synth.UNIFORM
    v = torch.from_numpy(w.vis()).cuda()
    plan0 = _plan(blink, w, warp_route=-1)
    assert plan0.query_i32(blink.Q_WARP_KERNEL) == 0
    ref = plan0.grid_image(v)
    uv = plan0.grid(v)
    ref_uv = plan0.image(uv)
    plan0.close()
    plan = _plan(blink, w)
    assert plan.query_i32(blink.Q_WARP_KERNEL) == 3
    img = torch.full(ref.shape, float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(v, img)
    peak = ref.abs().amax(dim=(-2, -1), keepdim=True)
    assert torch.isfinite(img).all()
    assert ((img - ref).abs() <= 1e-5 * peak).all()
    again = torch.full(ref.shape, float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(v, again)
    assert torch.equal(img, again)
    img_uv = torch.full(ref.shape, float("nan"), dtype=torch.float32, device="cuda")
    plan.image(uv, img_uv)
    assert torch.isfinite(img_uv).all()
    assert ((img_uv - ref_uv).abs() <= 1e-5 * peak).all()
    plan.close()


def test_corrections_fused_into_the_residue_column_pass(torch_cuda, blink):
    """f2 fused at load on the 2048^2 route: k_cols_res multiplies every visibility by the plan's factor as its
    lanes form their cells; against the stand-alone pass (blink_correct, then the plain call) on every pixel,
    and switching it off again restores the plain images bit for bit."""
    torch = torch_cuda
    w = synth.config_mwa2(n_t=2, n_ch=2)
    w.n_pix, w.pixscale = 2048, 30.0 * synth.ARCSEC
    rng = np.random.default_rng(23)
    n_ant = w.ant_enu_m.shape[0]
    gains = rng.uniform(0.5, 2.0, (w.n_ch, n_ant)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (w.n_ch, n_ant)))
    cables = rng.uniform(0.0, 300.0, n_ant)
    v = torch.from_numpy(w.vis()).cuda()
    plan = _plan(blink, w)
    assert plan.query_i32(blink.Q_WARP_KERNEL) == 3
    plain = plan.grid_image(v).clone()
    plan.set_corrections(gains, cables, 0.002, -0.001)
    ref = plan.grid_image(plan.correct(v)).clone()
    plan.apply_corrections(True)
    img = torch.full(ref.shape, float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(v, img)
    assert torch.isfinite(img).all()
    peak = ref.abs().amax(dim=(-2, -1), keepdim=True)
    assert ((img - ref).abs() <= 1e-5 * peak).all()
    assert not torch.equal(img, plain)
    plan.apply_corrections(False)
    assert torch.equal(plan.grid_image(v), plain)
    plan.close()


@pytest.mark.parametrize("n_pix,chunk_mb", [(4096, 64), (4096, 100), (2048, 40)])
def test_chunked_residue_column_pass(torch_cuda, blink, oracle, n_pix, chunk_mb):
    """The launch configuration bench.py times for mwa2: the two-kernel route cut into SEVERAL launch pairs
    (snap_base > 0 through k_cols_res + k_image_rows), forced on a small batch with blink_options.image_chunk_mb.
    9 snapshots of 3 channels; 64 MiB / 40 MiB give chunks of 2 snapshots (the channel wraps inside a chunk and
    across chunk boundaries), 100 MiB chunks of 3.  Through blink_grid_image AND blink_image, NaN-prefilled
    images, every snapshot against the oracle on sampled pixels, and bit-equal to the same plan run with the
    default 2 GB budget (one pair)."""
    torch = torch_cuda
    w = synth.config_mwa2(n_t=3, n_ch=3)
    if n_pix == 2048:
        w.n_pix, w.pixscale = 2048, 30.0 * synth.ARCSEC
    vis = w.vis()
    v = torch.from_numpy(vis).cuda()
    n, n_snap = w.n_pix, w.n_t * w.n_ch
    one = _plan(blink, w)
    assert one.query_i32(blink.Q_WARP_KERNEL) == 3 and one.query_i32(blink.Q_FUSED_PATH) == 0
    one.reserve(w.n_t)
    assert one.query_i32(blink.Q_FUSED_CHUNK) >= n_snap and one.query_i32(blink.Q_IMAGE_CHUNK) >= n_snap
    ref = one.grid_image(v)
    uv = one.grid(v)
    ref_uv = one.image(uv)
    one.close()
    plan = _plan(blink, w, image_chunk_mb=chunk_mb)
    plan.reserve(w.n_t)
    assert plan.query_i32(blink.Q_WARP_KERNEL) == 3 and plan.query_i32(blink.Q_FUSED_PATH) == 0
    chunk = plan.query_i32(blink.Q_FUSED_CHUNK)
    assert chunk == plan.query_i32(blink.Q_IMAGE_CHUNK)
    assert 1 <= chunk and 3 * chunk <= n_snap, f"chunk {chunk}: fewer than 3 launch pairs"
    if chunk_mb != 100:
        assert chunk % w.n_ch != 0                   # the channel of a chunk's first snapshot differs chunk to chunk
    img = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(v, img)
    img_uv = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.float32, device="cuda")
    plan.image(uv, img_uv)
    torch.cuda.synchronize()
    assert torch.isfinite(img).all() and torch.isfinite(img_uv).all(), "image not fully written"
    assert torch.equal(img, ref), "chunking changed blink_grid_image's result"
    assert torch.equal(img_uv, ref_uv), "chunking changed blink_image's result"
    imh, imh_uv = img.cpu().numpy().reshape(-1, n, n), img_uv.cpu().numpy().reshape(-1, n, n)
    yx = _pixels(n, 47)
    for s in range(n_snap):
        _sampled_pixel_check(oracle, w, vis, s, imh[s], yx)
        _sampled_pixel_check(oracle, w, vis, s, imh_uv[s], yx)
    plan.close()


def test_corrections_fused_into_the_residue_column_pass_against_oracle(torch_cuda, blink, oracle):
    """f2 fused at load on k_cols_res (2048^2), against the ORACLE chain (oracle/corrections.py in fp64 ->
    gridding -> weighting -> literal sums on sampled pixels), in two launch pairs."""
    torch = torch_cuda
    from oracle import corrections as oc
    w = synth.config_mwa2(n_t=2, n_ch=2)
    w.n_pix, w.pixscale = 2048, 30.0 * synth.ARCSEC
    rng = np.random.default_rng(29)
    n_ant = w.ant_enu_m.shape[0]
    gains = rng.uniform(0.5, 2.0, (w.n_ch, n_ant)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (w.n_ch, n_ant)))
    cables = rng.uniform(0.0, 300.0, n_ant)
    l0, m0 = 0.002, -0.001
    vis = w.vis()
    plan = _plan(blink, w, image_chunk_mb=40)
    plan.set_corrections(gains, cables, l0, m0)
    plan.apply_corrections(True)
    assert plan.query_i32(blink.Q_WARP_KERNEL) == 3 and plan.query_i32(blink.Q_CORR_FUSED) == 1
    n = w.n_pix
    img = torch.full((w.n_t, w.n_ch, n, n), float("nan"), dtype=torch.float32, device="cuda")
    plan.grid_image(torch.from_numpy(vis).cuda(), img)
    torch.cuda.synchronize()
    assert torch.isfinite(img).all()
    assert plan.query_i32(blink.Q_FUSED_CHUNK) < w.n_t * w.n_ch
    F_ref = oc.correction_factors(w.ant_enu_m, w.freq_hz, gains, cables, l0, m0)
    vis_c = oc.apply_corrections(vis, F_ref).astype(np.complex64)
    imh = img.cpu().numpy().reshape(-1, n, n)
    yx = _pixels(n, 53)
    for s in range(w.n_t * w.n_ch):
        _sampled_pixel_check(oracle, w, vis_c, s, imh[s], yx)
    plan.close()


@pytest.mark.parametrize("seed", [11, 12])
def test_residue_routes_on_random_arrays(torch_cuda, blink, seed):
    """The residue-class kernels (k_img1024r, k_cols_res) against the line kernels (warp_route = -1) on every
    pixel, for randomly drawn arrays: centrally condensed layouts of 24..128 antennas, some with a regular
    sub-array (many baselines per cell), pixel scales that put the longest baselines at 0.6..4 times the grid
    edge (dropped baselines), 1..3 channels and time steps, both weightings, N = 1024 / 2048 / 4096 -- through
    blink_grid_image and blink_image.  Configurations the routes do not apply to compare the line kernels
    with themselves."""
    torch = torch_cuda
    rng = np.random.default_rng(seed)
    applied = 0
    for _ in range(8):
        n_pix = int(rng.choice([1024, 1024, 2048, 4096]))
        n_ant = int(rng.integers(24, 129))
        ext = float(rng.choice([300.0, 800.0, 1500.0, 3000.0]))
        rad = np.minimum(rng.exponential(ext / 4, n_ant), ext)
        phi = rng.uniform(0, 2 * np.pi, n_ant)
        ant = np.stack([rad * np.cos(phi), rad * np.sin(phi), np.zeros(n_ant)], 1)
        if rng.random() < 0.3:
            ant[: n_ant // 4] = np.round(ant[: n_ant // 4] / 40.0) * 40.0
        n_ch, n_t = int(rng.integers(1, 4)), int(rng.integers(1, 4))
        f0 = float(rng.choice([120e6, 154e6, 200e6]))
        freq = f0 + 1e4 * np.arange(n_ch)
        frac = float(rng.choice([0.6, 0.9, 1.3, 2.5, 4.0]))
        pixscale = frac * 0.5 / (2 * ext * f0 / 299792458.0)
        weighting = int(rng.integers(0, 2))
        n_bl = n_ant * (n_ant - 1) // 2
        vis = (rng.standard_normal((n_t, n_ch, n_bl)) + 1j * rng.standard_normal((n_t, n_ch, n_bl))).astype(np.complex64)
        v = torch.from_numpy(vis).cuda()
        plan0 = blink.Plan(ant, freq, n_pix, pixscale, weighting, options=dict(warp_route=-1))
        ref, uv = plan0.grid_image(v), plan0.grid(v)
        ref_uv = plan0.image(uv)
        plan0.close()
        plan = blink.Plan(ant, freq, n_pix, pixscale, weighting)
        applied += plan.query_i32(blink.Q_WARP_KERNEL) in (2, 3)
        img = torch.full(ref.shape, float("nan"), dtype=torch.float32, device="cuda")
        plan.grid_image(v, img)
        img_uv = torch.full(ref.shape, float("nan"), dtype=torch.float32, device="cuda")
        plan.image(uv, img_uv)
        plan.close()
        peak = ref.abs().amax(dim=(-2, -1), keepdim=True).clamp_min(1e-30)
        assert torch.isfinite(img).all() and torch.isfinite(img_uv).all()
        assert ((img - ref).abs() <= 1e-5 * peak).all() and ((img_uv - ref_uv).abs() <= 1e-5 * peak).all()
        del v, ref, uv, ref_uv, img, img_uv
        torch.cuda.empty_cache()
    assert applied >= 3
