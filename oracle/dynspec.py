"""CPU ORACLE for the post-imaging transient front end.  TEST INFRASTRUCTURE ONLY.

Plain numpy, fp64, one explicit loop over time in the order of the text.  Shares no code with the CUDA
path (paper_2405_13478_b200/csrc/blink_dynspec.cu); only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it.

What the paper says (no formula is printed):
  * "imaging artefacts like side-lobes can be removed by subtracting a reference image of the same
    field (formed as a combination of previous images or prepared prior to the processing)"
    (PAPER.md:76);
  * "Such a reference image can be the preceding 'dirty image' image, some form of an average of the
    sequence of previous images recorded during the same observation or a model image";
  * "once the data cube of images (of multiple time steps and frequency channels) are created, dynamic
    spectra from all pixels (i.e time series in different directions in the sky) will be formed"
    (PAPER.md:84).

Readings (DESIGN.md c21-c23):
  c21  one recurrence covers the three references the text names.  Per channel and pixel, with the
       reference R_0 handed in (the state left by the previous batch, a model image, or zeros):
           D_t     = I_t - R_t
           R_{t+1} = (1 - alpha) R_t + alpha I_t
       alpha = 1: R_t = I_{t-1}, the preceding dirty image;  alpha = 0: R_t = R_0, a fixed model /
       prepared image;  0 < alpha < 1: an exponentially weighted average of the previous images
       ("some form of an average of the sequence of previous images").  The reference is built from
       the images themselves, not from the differences, and never includes the current image.
  c22  a dynamic spectrum is the (channel, time) plane of one pixel: the cube [t][ch][y][x] is
       transposed to [y][x][ch][t], time fastest (a time series per direction and channel).
  c23  the reference after the last image, R_{n_t}, is returned so that consecutive batches of one
       observation chain exactly like one long batch.
Parity vs the paper's own code: UNPINNED (this stage is described as planned work).
"""
from __future__ import annotations

import numpy as np


def dynamic_spectra(images, alpha, ref0=None):
    """images [n_t][n_ch][N][N] -> (dyn float64 [N][N][n_ch][n_t], ref_out float64 [n_ch][N][N])."""
    img = np.asarray(images, np.float64)
    n_t, n_ch, ny, nx = img.shape
    a = float(alpha)
    R = np.zeros((n_ch, ny, nx)) if ref0 is None else np.array(ref0, np.float64, copy=True)
    dyn = np.empty((ny, nx, n_ch, n_t), np.float64)
    for t in range(n_t):
        D = img[t] - R                               # c21: subtract the reference of this time step
        R = (1.0 - a) * R + a * img[t]               # c21: then fold the image into the reference
        for ch in range(n_ch):
            dyn[:, :, ch, t] = D[ch]                 # c22: pixel-major, time fastest
    return dyn, R
