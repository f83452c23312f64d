"""CPU ORACLE for the pre-gridding corrections (section 4.2, :142-156).  TEST INFRASTRUCTURE ONLY.

Plain numpy, fp64 / complex128, no blocking or reordering.  Shares no code with the CUDA path
(paper_2405_13478_b200/csrc/blink_correct.cu); only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it.

The paper names three corrections applied to the visibilities before imaging -- (i) cable-length
phase, (ii) calibration in phase and amplitude, (iii) geometric phase rotation of the phase centre
 -- and that antenna-level corrections "can be applied to visibilities
(post-correlation)" (:156), but prints no formula.  Readings (DESIGN.md c18-c20), chosen so that
they follow from the correlation product V_ij = E_i conj(E_j) (Eq. 2, with the
conjugate the extraction lost, reading c10) and Eq. 5's sign:

  c18  antenna model: the voltage of antenna i reaches the correlator as a_i(nu) E_i(nu) with
       a_i = g_i exp(-2 pi i nu L_i / c): g_i the calibration solution, L_i the electrical cable
       length (a delay L_i / c multiplies the spectrum by exp(-2 pi i nu tau)).  So the measured
       V_ij = a_i conj(a_j) V_ij(true) and the correction divides by a_i conj(a_j).
  c19  geometric phase: multiply by exp(+2 pi i (u l0 + v m0 + w (n0 - 1))), n0 = sqrt(1-l0^2-m0^2),
       (u, v, w) = (r_j - r_i) nu / c un-snapped, so that a source at (l0, m0), whose visibility is
       S exp(-2 pi i (u l0 + v m0 + w (n0 - 1))) (Eq. 4-5 PAPER.md:162-167 with the w term kept),
       becomes the constant S: it sits at the phase centre.
  c20  the three factors are combined in fp64 into one factor per (channel, baseline) and the
       visibilities are multiplied once.

Pins (tests/test_oracle_pins.py, -m "not gpu"): identity inputs give exactly 1; visibilities built
from per-antenna VOLTAGES with gains and cable delays (never touching this module's formula) are
restored to the ideal ones; a unit source at (l0, m0) becomes V = 1 on every baseline and images to
1.0 at the centre pixel; swapping two antennas conjugates the factor.
Parity vs the paper's own kernels: UNPINNED (no code, no formula in the text).
"""
from __future__ import annotations

import numpy as np

C_M_PER_S = 299792458.0


def correction_factors(ant_enu_m, freq_hz, gains=None, cable_len_m=None, l0=0.0, m0=0.0):
    """complex128 [n_ch][n_bl], baseline order bl(i,j), i < j, i-major (the boundary's order)."""
    ant = np.asarray(ant_enu_m, np.float64)
    freq = np.asarray(freq_hz, np.float64).reshape(-1)
    n_ant, n_ch = ant.shape[0], freq.shape[0]
    g = np.ones((n_ch, n_ant), np.complex128) if gains is None else np.asarray(gains, np.complex128)
    L = np.zeros(n_ant) if cable_len_m is None else np.asarray(cable_len_m, np.float64)
    n0 = np.sqrt(1.0 - l0 * l0 - m0 * m0)
    out = np.empty((n_ch, n_ant * (n_ant - 1) // 2), np.complex128)
    for ch in range(n_ch):
        sc = freq[ch] / C_M_PER_S
        a = g[ch] * np.exp(-2j * np.pi * sc * L)          # c18: a_i = g_i exp(-2 pi i nu L_i / c)
        bl = 0
        for i in range(n_ant - 1):
            j = np.arange(i + 1, n_ant)
            u = (ant[j, 0] - ant[i, 0]) * sc
            v = (ant[j, 1] - ant[i, 1]) * sc
            w = (ant[j, 2] - ant[i, 2]) * sc
            rot = np.exp(2j * np.pi * (u * l0 + v * m0 + w * (n0 - 1.0)))   # c19
            out[ch, bl:bl + len(j)] = rot / (a[i] * np.conj(a[j]))          # c18, c20
            bl += len(j)
    return out


def apply_corrections(vis, factors):
    """vis complex [n_t][n_ch][n_bl] -> complex128, vis * factors (one multiply per visibility)."""
    return np.asarray(vis, np.complex128) * np.asarray(factors, np.complex128)[None, :, :]
