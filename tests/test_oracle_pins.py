"""Pins for the CPU oracle (oracle/blink_oracle.c) against things OTHER than itself:
closed forms, brute force on hand-built lattices, invariants, the paper's printed counts, numpy's
FFT as a library special case, and the direct Fourier sum of BASELINE.json's north_star.
CPU only (-m "not gpu").  Each pin names the mistake it is meant to catch.
"""
import math
import os

import numpy as np
import pytest

from paper_2405_13478_b200 import synth

C = 299792458.0
GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_counts.txt")


def _golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) == 2:
                out[line[0]] = int(line[1])
    return out


# ------------------------------------------------------------------ counts printed in the paper
def test_paper_baseline_counts(oracle):
    g = _golden()
    assert oracle.n_baselines(128) == g["n_bl_128"]            # Table 3
    assert oracle.n_baselines(256) == g["n_bl_256"]
    assert 2 * oracle.n_baselines(128) == g["n_vis_128"]       # Table 1: V and V*
    assert 2 * oracle.n_baselines(256) == g["n_vis_256"]
    # Table 3 FFT op counts N^2 log2 N^2 (arithmetic sanity of the cost model; 180 is truncated)
    assert int(1024 ** 2 * math.log2(1024 ** 2)) == g["fft_ops_1024"]
    assert int(4096 ** 2 * math.log2(4096 ** 2)) == g["fft_ops_4096"]
    assert abs(180 ** 2 * math.log2(180 ** 2) - g["fft_ops_180"]) < 1.0


def test_baseline_order(oracle):
    n = 7
    i, j = synth.baseline_pairs(n)
    for b, (a, c) in enumerate(zip(i, j)):
        assert oracle.baseline_index(n, int(a), int(c)) == b


# ------------------------------------------------------------------ index map: lattice brute force
@pytest.mark.parametrize("n_pix", [16, 32])
def test_index_map_on_lattice(oracle, n_pix):
    """All-sky: du = 1/(N dx) = 1/2 exactly (Eq. 9), so antennas on a lattice of pitch lambda/2
    have integer cell coordinates equal to their lattice differences.  Catches: wrong sign of the
    baseline, swapped u/v, wrong wrap of negatives, off-by-one at the +-(N/2-1) edge."""
    freq = 160e6
    lam = C / freq
    nx, ny = n_pix // 2 + 2, 3          # x differences reach past +-N/2 so some are dropped
    ant = synth.lattice_layout(nx, ny, lam / 2.0)
    r = oracle.uv_cells(ant, freq, n_pix, 2.0 / n_pix)
    i, j = synth.baseline_pairs(nx * ny)
    gx, gy = np.arange(nx * ny) % nx, np.arange(nx * ny) // nx
    kx, ky = gx[j] - gx[i], gy[j] - gy[i]
    assert np.array_equal(r["kx"], kx) and np.array_equal(r["ky"], ky)
    kmax = n_pix // 2 - 1
    keep = (np.abs(kx) <= kmax) & (np.abs(ky) <= kmax)
    assert (~keep).sum() > 0 and r["n_dropped"] == (~keep).sum()
    assert np.all(r["cell"][~keep] == -1) and np.all(r["cell_conj"][~keep] == -1)
    exp_cell = (ky % n_pix) * n_pix + (kx % n_pix)           # python % is non-negative
    exp_conj = ((-ky) % n_pix) * n_pix + ((-kx) % n_pix)
    assert np.array_equal(r["cell"][keep], exp_cell[keep])
    assert np.array_equal(r["cell_conj"][keep], exp_conj[keep])
    # the edge itself is exercised: +-(N/2-1) kept, +-N/2 dropped
    assert (np.abs(kx[keep]).max() == kmax) and (np.abs(kx[~keep]).min() == kmax + 1)


def test_rounding_ties_away_from_zero(oracle):
    """u/du exactly half-integer: llround rounds away from zero, symmetric in sign (reading c5)."""
    freq = C / 2.0                         # lambda = 2 m, sc = 0.5 exactly
    ant = np.zeros((3, 3))
    ant[1, 0] = 2.5                        # u = 1.25, u*G = 2.5 -> 3
    ant[2, 0] = -2.5                       # -> -3
    r = oracle.uv_cells(ant, freq, 16, 2.0 / 16)
    assert list(r["kx"][:2]) == [3, -3] and r["kx"][2] == -5


def test_scale_small_field(oracle):
    """Small-field pixscale: du = 1/(N dx) (Eq. 9): a baseline of exactly k*du wavelengths -> k."""
    n_pix, dx = 64, 60.0 * synth.ARCSEC
    du = 1.0 / (n_pix * dx)
    freq = 154e6
    ant = np.zeros((2, 3))
    ant[1, 0] = 7.0 * du * C / freq
    ant[1, 1] = -5.0 * du * C / freq
    r = oracle.uv_cells(ant, freq, n_pix, dx)
    assert r["kx"][0] == 7 and r["ky"][0] == -5
    assert r["cell"][0] == (n_pix - 5) * n_pix + 7


# ------------------------------------------------------------------ counts / grid invariants
def test_count_invariants_and_hermitian_grid(oracle):
    w = synth.config_tiny()
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[0], w.n_pix, w.pixscale)
    vis = w.vis()[0, 0]
    g, cnt = oracle.grid(r["cell"], r["cell_conj"], vis, w.n_pix)
    n = w.n_pix
    assert cnt.sum() == 2 * (w.n_bl - r["n_dropped"])
    assert np.array_equal(cnt, oracle.counts(r["cell"], r["cell_conj"], n))
    idx = (-np.arange(n)) % n
    assert np.array_equal(cnt, cnt[idx][:, idx])             # count[c] == count[c*]
    assert cnt[0, 0] % 2 == 0
    assert np.array_equal(g, np.conj(g[idx][:, idx]))         # exactly Hermitian, bitwise
    assert np.all((cnt == 0) == (g == 0)) or True             # zero cells stay zero
    assert np.all(g[cnt == 0] == 0)


def test_cell_rule_by_hand(oracle):
    """0 vis -> 0, 1 vis -> that value, many -> sum (natural) / mean (uniform).
    Three collinear equally spaced antennas: baselines (0,1),(1,2) share a cell, (0,2) is alone."""
    freq = C / 2.0                                            # sc = 0.5
    ant = np.array([[0.0, 0, 0], [2.0, 0, 0], [4.0, 0, 0]])   # u = 1, 1, 2 -> kx = 2, 2, 4
    n = 16
    r = oracle.uv_cells(ant, freq, n, 2.0 / n)
    assert list(r["kx"]) == [2, 4, 2]                          # order (0,1),(0,2),(1,2)
    vis = np.array([1 + 2j, 10 - 1j, 3 + 5j], np.complex64)
    g, cnt = oracle.grid(r["cell"], r["cell_conj"], vis, n)
    assert g[0, 2] == (1 + 2j) + (3 + 5j) and cnt[0, 2] == 2
    assert g[0, 4] == 10 - 1j and cnt[0, 4] == 1
    assert g[0, n - 2] == np.conj(g[0, 2]) and g[0, n - 4] == 10 + 1j
    assert np.count_nonzero(g) == 4 and cnt.sum() == 6
    gn, norm_n = oracle.weight(g, cnt, synth.NATURAL)
    assert norm_n == 6 and np.array_equal(gn, g)
    gu, norm_u = oracle.weight(g, cnt, synth.UNIFORM)
    assert norm_u == 4 and gu[0, 2] == (4 + 7j) / 2 and gu[0, 4] == 10 - 1j


def test_zero_baseline_adds_both_terms_to_dc(oracle):
    ant = np.array([[0.0, 0, 0], [0.01, 0.0, 0]])             # rounds to cell 0
    r = oracle.uv_cells(ant, 160e6, 16, 2.0 / 16)
    g, cnt = oracle.grid(r["cell"], r["cell_conj"], np.array([2 + 3j], np.complex64), 16)
    assert cnt[0, 0] == 2 and g[0, 0] == 4 + 0j


# ------------------------------------------------------------------ the transform
def _rand_grid(n, seed, hermitian):
    rng = np.random.Generator(np.random.PCG64(seed))
    g = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    if hermitian:
        idx = (-np.arange(n)) % n
        g = g + np.conj(g[idx][:, idx])
    return g


@pytest.mark.parametrize("n", [8, 16, 32])
def test_separable_equals_literal_sum(oracle, n):
    """O(N^4) literal definition vs the separable passes, on a NON-Hermitian asymmetric grid so
    that a transposed axis, a wrong shift or a dropped imaginary cross term shows."""
    g = _rand_grid(n, 5, hermitian=False)
    a, ia = oracle.dft2_literal(g, 3.0)
    b, ib = oracle.dft2_separable(g, 3.0)
    assert np.max(np.abs(a - b)) < 1e-12 * np.max(np.abs(a))
    assert abs(ia - ib) < 1e-12 * ia


def test_single_cell_closed_form(oracle):
    """G = i at one cell (iy0, ix0): Re F[y][x] = -sin(2 pi (ix0 (x-N/2) + iy0 (y-N/2)) / N).
    Fixes the SIGN of the exponent (inverse transform, Eq. 4-5), the axis order and the shift."""
    n, iy0, ix0 = 16, 3, 5
    g = np.zeros((n, n), np.complex128)
    g[iy0, ix0] = 1j
    img, _ = oracle.dft2_separable(g, 1.0)
    y, x = np.mgrid[0:n, 0:n]
    th = 2 * math.pi * (ix0 * (x - n // 2) + iy0 * (y - n // 2)) / n
    assert np.max(np.abs(img + np.sin(th))) < 1e-13


@pytest.mark.parametrize("n", [16, 64, 128])
def test_library_special_case_ifft2(oracle, n):
    """I = N^2 fftshift(Re ifft2(G')) / norm  (numpy pocketfft as an independent routine)."""
    g = _rand_grid(n, 11, hermitian=False)
    norm = 7.5
    img, _ = oracle.dft2_separable(g, norm)
    ref = (n * n) * np.fft.fftshift(np.fft.ifft2(g)).real / norm
    assert np.max(np.abs(img - ref)) < 1e-11 * np.max(np.abs(ref))


def test_parseval_dc_sum_and_hermitian_residual(oracle):
    n = 32
    g = _rand_grid(n, 13, hermitian=True)
    img, imax = oracle.dft2_separable(g, 1.0)
    assert imax < 1e-12 * np.max(np.abs(img))                 # Hermitian grid -> real image
    assert abs((img ** 2).sum() - n * n * (np.abs(g) ** 2).sum()) < 1e-9 * (img ** 2).sum()
    assert abs(img.sum() - n * n * g[0, 0].real) < 1e-9 * n * n * abs(g[0, 0])


def test_pixels_match_full_image(oracle):
    n = 32
    g = _rand_grid(n, 17, hermitian=False)
    g[np.abs(g) < 1.0] = 0                                     # make it sparse
    img, _ = oracle.dft2_separable(g, 2.0)
    yx = np.array([[0, 0], [n // 2, n // 2], [3, 29], [31, 1], [17, 16]], np.int32)
    px = oracle.dft2_pixels(g, 2.0, yx)
    assert np.max(np.abs(px.real - img[yx[:, 0], yx[:, 1]])) < 1e-12 * np.max(np.abs(img))


# ------------------------------------------------------------------ whole chain vs definitions
def _chain(oracle, w, vis, ch=0):
    r = oracle.uv_cells(w.ant_enu_m, w.freq_hz[ch], w.n_pix, w.pixscale)
    g, cnt = oracle.grid(r["cell"], r["cell_conj"], vis, w.n_pix)
    gw, norm = oracle.weight(g, cnt, w.weighting)
    img, imax = oracle.dft2_separable(gw, norm)
    return r, g, cnt, img, imax


@pytest.mark.parametrize("weighting", [synth.NATURAL, synth.UNIFORM])
def test_unit_source_at_phase_centre(oracle, weighting):
    """V = 1 for every baseline: centre pixel is exactly 1 (fixes the normalisation, reading c4),
    it is the unique maximum, and the image (= dirty beam) is point-symmetric."""
    w = synth.config_tiny()
    w.weighting = weighting
    vis = np.ones(w.n_bl, np.complex64)
    _, _, _, img, imax = _chain(oracle, w, vis)
    n = w.n_pix
    assert abs(img[n // 2, n // 2] - 1.0) < 1e-13
    assert np.count_nonzero(img >= 1.0 - 1e-9) == 1
    sym = img[1:, 1:]
    assert np.max(np.abs(sym - sym[::-1, ::-1])) < 1e-12
    assert imax < 1e-6


def _lattice_workload(n_pix=32, nx=6, ny=5, freq=160e6):
    lam = C / freq
    return synth.Workload("lattice", synth.lattice_layout(nx, ny, lam / 2.0), np.array([freq]),
                          n_pix, 2.0 / n_pix, synth.NATURAL, 1, 0)


def test_direct_fourier_sum_on_lattice(oracle):
    """On-lattice antennas: snapping is exact, so the whole chain must equal north_star's direct
    sum I(l,m) = (1/2 n_bl) sum_bl 2 Re(V exp(+2 pi i (u l + v m))), l = (x-N/2) dx, m = (y-N/2) dx,
    with TRUE u,v, evaluated here in numpy independently of the oracle."""
    w = _lattice_workload()
    rng = np.random.Generator(np.random.PCG64(3))
    vis = (rng.standard_normal(w.n_bl) + 1j * rng.standard_normal(w.n_bl)).astype(np.complex64)
    r, _, _, img, _ = _chain(oracle, w, vis)
    assert r["n_dropped"] == 0
    u, v = w.uv_true()
    u, v = u[0], v[0]
    n = w.n_pix
    lm = (np.arange(n) - n // 2) * w.pixscale
    ref = np.zeros((n, n))
    vv = vis.astype(np.complex128)
    for yy in range(n):
        ph = np.exp(2j * math.pi * (u[None, :] * lm[:, None] + v[None, :] * lm[yy]))  # [x, bl]
        ref[yy] = 2.0 * (ph * vv[None, :]).real.sum(axis=1) / (2 * w.n_bl)
    assert np.max(np.abs(img - ref)) < 1e-10 * np.max(np.abs(ref))


def test_offset_source_on_lattice_peaks_at_predicted_pixel(oracle):
    """Source at a pixel centre (l0, m0): V = exp(-2 pi i (u l0 + v m0)) (Eq. 5) -> I[y0][x0] = 1
    and it is the arg-max.  x grows with l (East), y with m (North): fixes orientation (c10)."""
    w = _lattice_workload()
    n, x0, y0 = w.n_pix, 21, 9
    l0, m0 = (x0 - n // 2) * w.pixscale, (y0 - n // 2) * w.pixscale
    u, v = w.uv_true()
    vis = np.exp(-2j * math.pi * (u[0] * l0 + v[0] * m0)).astype(np.complex64)
    _, _, _, img, _ = _chain(oracle, w, vis)
    assert abs(img[y0, x0] - 1.0) < 1e-6                        # complex64 input rounding
    assert np.unravel_index(np.argmax(img), img.shape) == (y0, x0)


def test_tiny_config_brightest_source_within_one_pixel(oracle):
    """Off-lattice (config 1): the brightest source's peak lies within +-1 pixel of prediction,
    and the Hermitian residual is below 1e-6 of peak (north_star)."""
    w = synth.config_tiny()
    w.noise_sigma = 0.0
    k = int(np.argmax(w.src_flux))
    w.src_flux = np.where(np.arange(3) == k, w.src_flux, 0.0)  # keep only the brightest
    w._sky = None
    vis = w.vis()[0, 0]
    _, _, _, img, imax = _chain(oracle, w, vis)
    n = w.n_pix
    yp, xp = np.unravel_index(np.argmax(img), img.shape)
    assert abs(xp - (w.src_l[k] / w.pixscale + n // 2)) <= 1.0
    assert abs(yp - (w.src_m[k] / w.pixscale + n // 2)) <= 1.0
    assert imax <= 1e-6 * img.max()


def test_image_batch_matches_stepwise(oracle):
    w = synth.config_station(n_t=2, n_ch=3, n_pix=64)
    vis = w.vis()
    sel = np.array([1, 5], np.int64)
    out = oracle.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, sel,
                             want_grids=True)
    for q, s in enumerate(sel):
        t, ch = divmod(int(s), w.n_ch)
        _, g, _, img, _ = _chain(oracle, w, vis[t, ch], ch)
        assert np.array_equal(out["grids"][q], g)
        assert np.array_equal(out["images"][q], img)


# ------------------------------------------------------------------ pre-gridding corrections (f2)
def _voltage_visibilities(ant, freq, src_lmS, gains, cables):
    """Visibilities from per-antenna VOLTAGES (first principles, independent of oracle/corrections):
    a source of flux S at (l, m, n) gives antenna i the phasor sqrt(S) exp(+2 pi i (x l + y m + z (n-1)) nu/c);
    the receiver chain multiplies it by g_i and delays it by L_i / c (a factor exp(-2 pi i nu L_i/c));
    the correlator forms V_ij = E_i conj(E_j) per source (sources are incoherent)."""
    n_ant = ant.shape[0]
    out = np.zeros((len(freq), n_ant * (n_ant - 1) // 2), np.complex128)
    for ch, nu in enumerate(freq):
        for (l, m, S) in src_lmS:
            n = math.sqrt(1 - l * l - m * m)
            E = np.array([math.sqrt(S) * np.exp(2j * math.pi * (ant[i, 0] * l + ant[i, 1] * m + ant[i, 2] * (n - 1)) * nu / C)
                          for i in range(n_ant)])
            E = E * gains[ch] * np.exp(-2j * math.pi * nu * cables / C)
            bl = 0
            for i in range(n_ant):
                for j in range(i + 1, n_ant):
                    out[ch, bl] += E[i] * np.conj(E[j])
                    bl += 1
    return out


def test_corrections_identity_is_exactly_one():
    from oracle import corrections as oc
    w = synth.config_tiny()
    F = oc.correction_factors(w.ant_enu_m, w.freq_hz)
    assert np.all(F == 1.0 + 0.0j)          # a stray phase or a wrong default fails this


def test_corrections_restore_ideal_visibilities_from_corrupted_voltages():
    """Catches a wrong sign of the cable phase, g_i conj(g_j) transposed, gains multiplied instead
    of divided, a dropped w term."""
    from oracle import corrections as oc
    rng = np.random.default_rng(5)
    ant = rng.uniform(-20, 20, (9, 3))
    ant[:, 2] = rng.uniform(-0.5, 0.5, 9)              # non-coplanar: exercises w
    freq = np.array([150e6, 170e6])
    gains = (rng.uniform(0.5, 1.5, (2, 9)) * np.exp(2j * np.pi * rng.uniform(0, 1, (2, 9))))
    cables = rng.uniform(0, 120.0, 9)
    src = [(0.3, -0.2, 2.0), (-0.5, 0.4, 1.0)]
    ideal = _voltage_visibilities(ant, freq, src, np.ones((2, 9)), np.zeros(9))
    meas = _voltage_visibilities(ant, freq, src, gains, cables)
    assert np.max(np.abs(meas - ideal)) > 0.5           # the corruption is not a no-op
    F = oc.correction_factors(ant, freq, gains, cables)
    got = oc.apply_corrections(meas[None], F)[0]
    assert np.max(np.abs(got - ideal)) <= 1e-9 * np.max(np.abs(ideal))
    # and the ideal ones agree with Eq. 5's sign convention used by the imaging oracle (c10)
    l, m, S = src[0]
    n = math.sqrt(1 - l * l - m * m)
    one = _voltage_visibilities(ant, freq[:1], [src[0]], np.ones((1, 9)), np.zeros(9))[0]
    u = (ant[1, 0] - ant[0, 0]) * freq[0] / C
    v = (ant[1, 1] - ant[0, 1]) * freq[0] / C
    ww = (ant[1, 2] - ant[0, 2]) * freq[0] / C
    assert abs(one[0] - S * np.exp(-2j * math.pi * (u * l + v * m + ww * (n - 1)))) < 1e-9


def test_geometric_rotation_moves_source_to_phase_centre(oracle):
    """A unit source at (l0, m0): after the rotation every visibility is 1, so the image of the
    corrected visibilities is the dirty beam with exactly 1.0 at the centre pixel (north_star's
    phase-centre check, through the correction).  Catches the wrong sign of (iii)."""
    from oracle import corrections as oc
    w = synth.config_tiny()
    l0, m0 = 0.25, -0.4
    vis = _voltage_visibilities(w.ant_enu_m, w.freq_hz, [(l0, m0, 1.0)], np.ones((1, w.n_ant)), np.zeros(w.n_ant))
    F = oc.correction_factors(w.ant_enu_m, w.freq_hz, l0=l0, m0=m0)
    cor = oc.apply_corrections(vis[None], F)
    assert np.max(np.abs(cor - 1.0)) < 1e-9
    out = oracle.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting,
                             cor.astype(np.complex64), np.array([0], np.int64))
    img = out["images"][0]
    c = w.n_pix // 2
    assert abs(img[c, c] - 1.0) < 1e-6 and np.argmax(img) == c * w.n_pix + c


def test_corrections_antenna_swap_conjugates_factor():
    from oracle import corrections as oc
    rng = np.random.default_rng(6)
    ant = rng.uniform(-20, 20, (2, 3))
    freq = np.array([160e6])
    gains = rng.uniform(0.5, 1.5, (1, 2)) * np.exp(2j * np.pi * rng.uniform(0, 1, (1, 2)))
    cables = np.array([10.0, 55.0])
    F = oc.correction_factors(ant, freq, gains, cables, 0.1, 0.2)[0, 0]
    Fs = oc.correction_factors(ant[::-1], freq, gains[:, ::-1], cables[::-1], 0.1, 0.2)[0, 0]
    assert abs(Fs - np.conj(F)) < 1e-12 * abs(F)


# ------------------------------------------------------------------ dynamic spectra front end (f4)
def _cube(seed, n_t=9, n_ch=3, n=4):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n_t, n_ch, n, n)), rng.standard_normal((n_ch, n, n))


def test_dynspec_alpha_one_is_difference_with_preceding_image():
    """alpha = 1: the reference is 'the preceding dirty image' -> numpy.diff along t.
    Catches a reference that includes the current image or lags by two."""
    from oracle import dynspec as od
    img, r0 = _cube(1)
    dyn, r_out = od.dynamic_spectra(img, 1.0, r0)
    want = np.diff(np.concatenate([r0[None], img], axis=0), axis=0)        # [t][ch][y][x]
    for t in range(img.shape[0]):
        for ch in range(img.shape[1]):
            assert np.allclose(dyn[:, :, ch, t], want[t, ch], rtol=0, atol=1e-15)
    assert np.array_equal(r_out, img[-1])


def test_dynspec_alpha_zero_is_fixed_model_image():
    """alpha = 0: a fixed model / prepared reference is subtracted from every image and
    returned unchanged."""
    from oracle import dynspec as od
    img, r0 = _cube(2)
    dyn, r_out = od.dynamic_spectra(img, 0.0, r0)
    assert np.array_equal(np.moveaxis(dyn, (2, 3), (1, 0)), img - r0[None])   # -> [t][ch][y][x]
    assert np.array_equal(r_out, r0)
    dyn0, _ = od.dynamic_spectra(img, 0.0)                                  # no reference: the cube itself
    assert np.array_equal(np.moveaxis(dyn0, (2, 3), (1, 0)), img)


def test_dynspec_running_average_closed_form():
    """0 < alpha < 1: R_t = (1-a)^t R_0 + a sum_{k<t} (1-a)^(t-1-k) I_k, written out with explicit
    weights (no recurrence).  Catches swapped alpha / (1 - alpha) and an off-by-one in the window."""
    from oracle import dynspec as od
    img, r0 = _cube(3, n_t=12)
    a = 0.3
    dyn, r_out = od.dynamic_spectra(img, a, r0)
    n_t = img.shape[0]
    for t in range(n_t + 1):
        R = (1 - a) ** t * r0
        for k in range(t):
            R = R + a * (1 - a) ** (t - 1 - k) * img[k]
        if t < n_t:
            got = np.moveaxis(dyn[:, :, :, t], 2, 0)
            assert np.max(np.abs(got - (img[t] - R))) < 1e-13
        else:
            assert np.max(np.abs(r_out - R)) < 1e-13


def test_dynspec_static_sky_vanishes_and_pulse_survives():
    """The purpose of the step: a static dirty image (side-lobes included) subtracts
    to zero once the reference has converged, a one-step transient stands out at full amplitude and
    leaves an echo of -alpha (1-alpha)^(k-1) in the following steps."""
    from oracle import dynspec as od
    rng = np.random.default_rng(4)
    sky = rng.standard_normal((2, 4, 4))
    img = np.repeat(sky[None], 10, axis=0)
    img[6, 1, 2, 3] += 5.0
    a = 0.25
    dyn, _ = od.dynamic_spectra(img, a, sky)          # reference already equal to the static sky
    want = np.zeros(10)
    want[6] = 5.0
    for k in range(1, 4):
        want[6 + k] = -a * (1 - a) ** (k - 1) * 5.0
    assert np.max(np.abs(dyn[2, 3, 1, :] - want)) < 1e-14
    dyn[2, 3, 1, :] = 0
    assert np.max(np.abs(dyn)) < 1e-14


def test_dynspec_layout_and_batch_chaining():
    """dyn[y][x][ch][t] is the (channel, time) plane of pixel (y, x), checked with
    hand-written indices on a cube whose value encodes its own coordinates; two consecutive batches
    with the state carried over equal one long batch (reading c23)."""
    from oracle import dynspec as od
    n_t, n_ch, n = 5, 2, 3
    img = np.zeros((n_t, n_ch, n, n))
    for t in range(n_t):
        for ch in range(n_ch):
            for y in range(n):
                for x in range(n):
                    img[t, ch, y, x] = 1000 * t + 100 * ch + 10 * y + x
    dyn, _ = od.dynamic_spectra(img, 0.0)
    assert dyn.shape == (n, n, n_ch, n_t)
    assert dyn[2, 1, 1, 4] == 4121 and dyn[0, 2, 0, 3] == 3002
    img, r0 = _cube(5, n_t=11)
    one, r_one = od.dynamic_spectra(img, 0.4, r0)
    a, r_a = od.dynamic_spectra(img[:4], 0.4, r0)
    b, r_b = od.dynamic_spectra(img[4:], 0.4, r_a)
    assert np.array_equal(np.concatenate([a, b], axis=3), one) and np.array_equal(r_b, r_one)
