"""ctypes wrapper around oracle/blink_oracle.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It shares nothing with paper_2405_13478_b200 (the CUDA path) and imports nothing from it.
All arithmetic lives in blink_oracle.c (fp64, step-by-step from PAPER.md, see that file's header);
this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "blink_oracle.c")
_LIB = os.path.join(_HERE, "libblink_oracle.so")
_lib = None

NATURAL, UNIFORM = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction: -ffp-contract=off)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-Wall", "-ffp-contract=off", "-fopenmp", "-shared",
               "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    c_dp = ctypes.POINTER(ctypes.c_double)
    c_fp = ctypes.POINTER(ctypes.c_float)
    c_i32p = ctypes.POINTER(ctypes.c_int32)
    c_i64p = ctypes.POINTER(ctypes.c_int64)
    c_u32p = ctypes.POINTER(ctypes.c_uint32)
    lib.oracle_n_baselines.restype = ctypes.c_int64
    lib.oracle_n_baselines.argtypes = [ctypes.c_int]
    lib.oracle_baseline_index.restype = ctypes.c_int64
    lib.oracle_baseline_index.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int]
    lib.oracle_uv_cells.restype = ctypes.c_int64
    lib.oracle_uv_cells.argtypes = [c_dp, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                    ctypes.c_double, c_i64p, c_i64p, c_i32p, c_i32p]
    lib.oracle_grid.restype = None
    lib.oracle_grid.argtypes = [c_i32p, c_i32p, ctypes.c_int64, c_fp, ctypes.c_int, c_dp, c_u32p]
    lib.oracle_counts.restype = None
    lib.oracle_counts.argtypes = [c_i32p, c_i32p, ctypes.c_int64, ctypes.c_int, c_u32p]
    lib.oracle_weight.restype = ctypes.c_double
    lib.oracle_weight.argtypes = [c_dp, c_u32p, ctypes.c_int, ctypes.c_int]
    for name in ("oracle_dft2_literal", "oracle_dft2_separable"):
        f = getattr(lib, name)
        f.restype = ctypes.c_int
        f.argtypes = [c_dp, ctypes.c_int, ctypes.c_double, c_dp, c_dp]
    lib.oracle_dft2_pixels.restype = ctypes.c_int
    lib.oracle_dft2_pixels.argtypes = [c_dp, ctypes.c_int, ctypes.c_double, c_i32p, ctypes.c_int64,
                                       c_dp, c_dp]
    lib.oracle_image_batch.restype = ctypes.c_int
    lib.oracle_image_batch.argtypes = [c_dp, ctypes.c_int, c_dp, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_double, ctypes.c_int, c_fp, c_i64p, ctypes.c_int64,
                                       c_dp, c_dp, ctypes.c_int]
    _lib = lib
    return lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def n_baselines(n_ant: int) -> int:
    return int(_load().oracle_n_baselines(n_ant))


def baseline_index(n_ant: int, i: int, j: int) -> int:
    return int(_load().oracle_baseline_index(n_ant, i, j))


def uv_cells(ant_enu_m, freq_hz: float, n_pix: int, pixscale: float):
    """Steps 1-3 for one channel -> dict(kx, ky, cell, cell_conj, n_dropped)."""
    lib = _load()
    ant = np.ascontiguousarray(ant_enu_m, dtype=np.float64)
    n_ant = ant.shape[0]
    n_bl = n_baselines(n_ant)
    kx = np.empty(n_bl, np.int64)
    ky = np.empty(n_bl, np.int64)
    cell = np.empty(n_bl, np.int32)
    cellc = np.empty(n_bl, np.int32)
    nd = lib.oracle_uv_cells(_p(ant, ctypes.c_double), n_ant, float(freq_hz), int(n_pix),
                             float(pixscale), _p(kx, ctypes.c_int64), _p(ky, ctypes.c_int64),
                             _p(cell, ctypes.c_int32), _p(cellc, ctypes.c_int32))
    if nd < 0:
        raise ValueError("oracle_uv_cells: bad arguments")
    return dict(kx=kx, ky=ky, cell=cell, cell_conj=cellc, n_dropped=int(nd))


def grid(cell, cell_conj, vis, n_pix: int):
    """Step 4 for one snapshot -> (grid complex128 [N,N] FFT-native order, count uint32 [N,N])."""
    lib = _load()
    cell = np.ascontiguousarray(cell, np.int32)
    cellc = np.ascontiguousarray(cell_conj, np.int32)
    v = np.ascontiguousarray(vis, dtype=np.complex64)
    assert v.shape == cell.shape
    g = np.empty((n_pix, n_pix), np.complex128)
    cnt = np.empty((n_pix, n_pix), np.uint32)
    lib.oracle_grid(_p(cell, ctypes.c_int32), _p(cellc, ctypes.c_int32), cell.shape[0],
                    _p(v.view(np.float32), ctypes.c_float), int(n_pix),
                    _p(g.view(np.float64), ctypes.c_double), _p(cnt, ctypes.c_uint32))
    return g, cnt


def counts(cell, cell_conj, n_pix: int):
    lib = _load()
    cell = np.ascontiguousarray(cell, np.int32)
    cellc = np.ascontiguousarray(cell_conj, np.int32)
    cnt = np.empty((n_pix, n_pix), np.uint32)
    lib.oracle_counts(_p(cell, ctypes.c_int32), _p(cellc, ctypes.c_int32), cell.shape[0],
                      int(n_pix), _p(cnt, ctypes.c_uint32))
    return cnt


def weight(grid_c128, count, weighting: int):
    """Step 5 -> (weighted grid copy, norm)."""
    lib = _load()
    g = np.array(grid_c128, dtype=np.complex128, order="C", copy=True)
    cnt = np.ascontiguousarray(count, np.uint32)
    norm = lib.oracle_weight(_p(g.view(np.float64), ctypes.c_double), _p(cnt, ctypes.c_uint32),
                             g.shape[0], int(weighting))
    return g, float(norm)


def _dft2(fname, grid_c128, norm):
    lib = _load()
    g = np.ascontiguousarray(grid_c128, np.complex128)
    n = g.shape[0]
    img = np.empty((n, n), np.float64)
    imax = ctypes.c_double(0.0)
    rc = getattr(lib, fname)(_p(g.view(np.float64), ctypes.c_double), n, float(norm),
                             _p(img, ctypes.c_double), ctypes.byref(imax))
    if rc != 0:
        raise MemoryError(fname)
    return img, float(imax.value)


def dft2_literal(grid_c128, norm):
    """Step 6, O(N^4) literal double sum -> (image fp64 [N,N], max|Im|)."""
    return _dft2("oracle_dft2_literal", grid_c128, norm)


def dft2_separable(grid_c128, norm):
    """Step 6, separable naive DFT -> (image fp64 [N,N], max|Im|)."""
    return _dft2("oracle_dft2_separable", grid_c128, norm)


def dft2_pixels(grid_c128, norm, yx):
    """Step 6 at listed (y, x) pixels only -> complex128 [n] (real part is the image value)."""
    lib = _load()
    g = np.ascontiguousarray(grid_c128, np.complex128)
    yx = np.ascontiguousarray(yx, np.int32).reshape(-1, 2)
    re = np.empty(yx.shape[0], np.float64)
    im = np.empty(yx.shape[0], np.float64)
    rc = lib.oracle_dft2_pixels(_p(g.view(np.float64), ctypes.c_double), g.shape[0], float(norm),
                                _p(yx, ctypes.c_int32), yx.shape[0], _p(re, ctypes.c_double),
                                _p(im, ctypes.c_double))
    if rc != 0:
        raise MemoryError("oracle_dft2_pixels")
    return re + 1j * im


def image_batch(ant_enu_m, freq_hz, n_pix, pixscale, weighting, vis, sel, want_grids=False,
                want_images=True, n_threads=0):
    """Whole chain for the snapshots `sel` (flat t*n_ch+ch) of vis [n_t, n_ch, n_bl] complex64.

    Returns dict(grids complex128 [n_sel,N,N] | None, images fp64 [n_sel,N,N] | None, threads).
    """
    lib = _load()
    ant = np.ascontiguousarray(ant_enu_m, np.float64)
    fr = np.ascontiguousarray(freq_hz, np.float64)
    v = np.ascontiguousarray(vis, np.complex64)
    assert v.ndim == 3 and v.shape[1] == fr.shape[0]
    sel = np.ascontiguousarray(sel, np.int64)
    n_sel = sel.shape[0]
    grids = np.empty((n_sel, n_pix, n_pix), np.complex128) if want_grids else None
    imgs = np.empty((n_sel, n_pix, n_pix), np.float64) if want_images else None
    rc = lib.oracle_image_batch(
        _p(ant, ctypes.c_double), ant.shape[0], _p(fr, ctypes.c_double), fr.shape[0], int(n_pix),
        float(pixscale), int(weighting), _p(v.view(np.float32), ctypes.c_float),
        _p(sel, ctypes.c_int64), n_sel,
        _p(grids.view(np.float64), ctypes.c_double) if want_grids else None,
        _p(imgs, ctypes.c_double) if want_images else None, int(n_threads))
    if rc < 0:
        raise RuntimeError("oracle_image_batch failed")
    return dict(grids=grids, images=imgs, threads=int(rc))
