"""Thin Python binding over the C-ABI library libblink.so (include/blink.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the C ABI.
PyTorch is used for device memory and streams, nothing else.  There is no fallback of any kind: if
libblink.so is missing or was not built, importing/using this module raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libblink.so")

NATURAL, UNIFORM = 0, 1
OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, ERESERVE, ECAPACITY = 0, -1, -2, -3, -4, -5, -6
STATIC_SCRATCH_BYTES = 32 << 20     # BLINK_STATIC_SCRATCH_BYTES
(Q_N_ANT, Q_N_BL, Q_N_CH, Q_N_PIX, Q_N_DROPPED, Q_WSUM, Q_N_OCC, Q_BBOX, Q_NORM, Q_CELL_IDX,
 Q_COUNTS, Q_IMAGE_PATH, Q_SCRATCH_BYTES, Q_IMAGE_CHUNK, Q_FUSED_PATH, Q_FUSED_CHUNK, Q_CORR, Q_CORR_FUSED,
 Q_TENSOR_ROUTE, Q_WARP_KERNEL, Q_FUSED_NZ, Q_FUSED_D) = range(22)

# include/blink.h (the product ABI) and include/blink_testing.h (host-only test hooks)
EXPORTS = ["blink_version", "blink_strerror", "blink_last_cuda_error", "blink_plan_create", "blink_plan_create_opts",
           "blink_plan_destroy", "blink_plan_query", "blink_plan_read", "blink_plan_reserve",
           "blink_grid", "blink_grid_image", "blink_plan_set_corrections", "blink_correct", "blink_dynspec",
           "blink_image", "blink_grid_validate", "blink_grid_image_host", "blink_plan_reserve_host",
           "blink_plan_apply_corrections", "blink_plan_refresh", "blink_image_static"]
TESTING_EXPORTS = ["blink_host_build_gather", "blink_host_fused_emulate", "blink_host_residue_emulate", "blink_probe_fp32"]


class Options(ctypes.Structure):
    """blink_options (include/blink.h): zero = let the plan decide."""
    _fields_ = [("struct_size", ctypes.c_int32), ("fused_route", ctypes.c_int32), ("polyphase", ctypes.c_int32),
                ("warp_route", ctypes.c_int32), ("warp_ring", ctypes.c_int32), ("grid_ring", ctypes.c_int32),
                ("grid_ring_min_snap", ctypes.c_int32), ("image_chunk_mb", ctypes.c_int32),
                ("tune", ctypes.c_int32 * 8)]

    def __init__(self, **kw):
        super().__init__()
        self.struct_size = ctypes.sizeof(Options)
        for k, v in kw.items():
            if k == "tune":
                for i, t in dict(v).items():
                    self.tune[int(i)] = int(t)
            else:
                if not hasattr(self, k):
                    raise TypeError(f"unknown blink option {k}")
                setattr(self, k, int(v))

_lib = None
_tlib = None
TESTING_LIB_PATH = os.path.join(_HERE, "libblink_testing.so")


class BlinkError(RuntimeError):
    def __init__(self, status: int, what: str):
        lib = load()
        msg = lib.blink_strerror(status).decode()
        cuda = lib.blink_last_cuda_error().decode()
        super().__init__(f"{what}: {msg} ({status})" + (f" [{cuda}]" if cuda else ""))
        self.status = status


def load() -> ctypes.CDLL:
    """dlopen libblink.so (raises if it has not been built; there is no other path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2405_13478_b200.build` "
                          "(nvcc, sm_100a); there is no CPU or PyTorch fallback")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    lib.blink_version.restype = ci
    lib.blink_strerror.restype = ctypes.c_char_p
    lib.blink_strerror.argtypes = [ci]
    lib.blink_last_cuda_error.restype = ctypes.c_char_p
    lib.blink_plan_create.restype = ci
    lib.blink_plan_create.argtypes = [ctypes.POINTER(vp), vp, ci, vp, ci, ci, cd, ci, vp]
    lib.blink_plan_create_opts.restype = ci
    lib.blink_plan_create_opts.argtypes = [ctypes.POINTER(vp), vp, ci, vp, ci, ci, cd, ci, vp, ctypes.POINTER(Options)]
    lib.blink_grid_validate.restype = ci
    lib.blink_grid_validate.argtypes = [vp, vp, ci, ctypes.POINTER(ctypes.c_int64), vp]
    lib.blink_grid_image_host.restype = ci
    lib.blink_grid_image_host.argtypes = [vp, vp, ci, vp, vp]
    lib.blink_plan_reserve_host.restype = ci
    lib.blink_plan_reserve_host.argtypes = [vp, ci]
    lib.blink_plan_refresh.restype = ci
    lib.blink_plan_refresh.argtypes = [vp, vp, vp]
    lib.blink_plan_destroy.restype = ci
    lib.blink_plan_destroy.argtypes = [vp]
    lib.blink_plan_query.restype = ci
    lib.blink_plan_query.argtypes = [vp, ci, ci, vp]
    lib.blink_plan_read.restype = ci
    lib.blink_plan_read.argtypes = [vp, ci, ci, vp, ctypes.c_size_t]
    lib.blink_plan_reserve.restype = ci
    lib.blink_plan_reserve.argtypes = [vp, ci]
    lib.blink_grid.restype = ci
    lib.blink_grid.argtypes = [vp, vp, ci, vp, vp]
    lib.blink_image.restype = ci
    lib.blink_image.argtypes = [vp, vp, ci, vp, vp]
    lib.blink_image_static.restype = ci
    lib.blink_image_static.argtypes = [vp, vp, ci, vp, vp]
    lib.blink_grid_image.restype = ci
    lib.blink_grid_image.argtypes = [vp, vp, ci, vp, vp]
    lib.blink_plan_set_corrections.restype = ci
    lib.blink_plan_set_corrections.argtypes = [vp, vp, vp, ctypes.c_double, ctypes.c_double, vp]
    lib.blink_plan_apply_corrections.restype = ci
    lib.blink_plan_apply_corrections.argtypes = [vp, ci, vp]
    lib.blink_correct.restype = ci
    lib.blink_correct.argtypes = [vp, vp, ci, vp, vp]
    lib.blink_dynspec.restype = ci
    lib.blink_dynspec.argtypes = [vp, vp, ci, ctypes.c_double, vp, vp, vp]
    _lib = lib
    return lib


def load_testing() -> ctypes.CDLL:
    """dlopen libblink_testing.so: the test hooks of include/blink_testing.h (host models of the table walks,
    the fp32 peak probe).  They are NOT in libblink.so -- the product library has no CPU model of anything."""
    global _tlib
    if _tlib is not None:
        return _tlib
    if not os.path.exists(TESTING_LIB_PATH):
        raise ImportError(f"{TESTING_LIB_PATH} not found: run `python -m paper_2405_13478_b200.build`")
    lib = ctypes.CDLL(TESTING_LIB_PATH)
    vp, ci = ctypes.c_void_p, ctypes.c_int
    lib.blink_strerror.restype = ctypes.c_char_p
    lib.blink_strerror.argtypes = [ci]
    lib.blink_last_cuda_error.restype = ctypes.c_char_p
    lib.blink_probe_fp32.restype = ci
    lib.blink_probe_fp32.argtypes = [ci, ci, vp, ctypes.c_size_t, ctypes.POINTER(ctypes.c_int64), vp]
    lib.blink_host_build_gather.restype = ci
    lib.blink_host_build_gather.argtypes = [vp, ci, ci, vp, vp, vp, vp]
    lib.blink_host_fused_emulate.restype = ci
    lib.blink_host_fused_emulate.argtypes = [vp, ci, ci, ci, vp, vp, vp]
    lib.blink_host_residue_emulate.restype = ci
    lib.blink_host_residue_emulate.argtypes = [vp, ci, ci, ci, vp, ci, vp, vp, vp]
    _tlib = lib
    return lib


def _check(status: int, what: str):
    if status != OK:
        raise BlinkError(status, what)


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def host_build_gather(cell: np.ndarray, n_pix: int):
    """blink_host_build_gather: cell-sorted gather tables of one channel (host logic, no GPU)."""
    lib = load_testing()
    cell = np.ascontiguousarray(cell, np.int32)
    n_bl = cell.shape[0]
    n_can = ctypes.c_int32(0)
    can_cell = np.zeros(max(n_bl, 1), np.int32)
    seg = np.zeros(n_bl + 1, np.int32)
    src = np.zeros(max(n_bl, 1), np.int32)
    rc = lib.blink_host_build_gather(cell.ctypes.data, n_bl, int(n_pix), ctypes.byref(n_can),
                                     can_cell.ctypes.data, seg.ctypes.data, src.ctypes.data)
    if rc < 0:
        raise BlinkError(rc, "blink_host_build_gather")
    n = n_can.value
    return dict(n_kept=rc, n_can=n, can_cell=can_cell[:n], seg_start=seg[:n + 1], src=src[:rc])


def host_fused_emulate(cell: np.ndarray, n_pix: int, chunk_vis: int, vis: np.ndarray):
    """blink_host_fused_emulate: phase S of the shared-memory route walked on the host (no GPU)."""
    lib = load_testing()
    cell = np.ascontiguousarray(cell, np.int32)
    vis = np.ascontiguousarray(vis, np.complex64)
    n_bl = cell.shape[0]
    sums = np.zeros(max(n_bl, 1), np.complex64)
    stats = np.zeros(3, np.int32)
    rc = lib.blink_host_fused_emulate(cell.ctypes.data, n_bl, int(n_pix), int(chunk_vis), vis.ctypes.data,
                                      sums.ctypes.data, stats.ctypes.data)
    if rc < 0:
        raise BlinkError(rc, "blink_host_fused_emulate")
    return dict(sums=sums[:stats[0]], n_can=int(stats[0]), groups=int(stats[1]), rows=int(stats[2]))


def host_residue_emulate(cell: np.ndarray, n_pix: int, weighting: int, vis: np.ndarray, units):
    """blink_host_residue_emulate: the residue-class kernels (N = 1024: k_img1024r; 2048 / 4096: k_cols_res +
    plain row sums) walked on the host (no GPU); returns the image rows of the listed units as
    {row index: float32[n_pix]}."""
    lib = load_testing()
    cell = np.ascontiguousarray(cell, np.int32)
    vis = np.ascontiguousarray(vis, np.complex64)
    units = np.ascontiguousarray(units, np.int32)
    per = 16 if n_pix == 1024 else 8
    rows = np.zeros((len(units), per, n_pix), np.float32)
    stats = np.zeros(3, np.int32)
    rc = lib.blink_host_residue_emulate(cell.ctypes.data, cell.shape[0], int(n_pix), int(weighting), vis.ctypes.data,
                                        len(units), units.ctypes.data, rows.ctypes.data, stats.ctypes.data)
    if rc < 0:
        raise BlinkError(rc, "blink_host_residue_emulate")
    out = {}
    for i, r in enumerate(units):
        for q in range(per):
            if n_pix == 1024:
                out[64 * (q % 8) + int(r) + (512 if q >= 8 else 0)] = rows[i, q]
            else:
                out[(n_pix // 8) * q + int(r)] = rows[i, q]
    return dict(rows=out, positions=int(stats[0]), longest_list=int(stats[1]), n_can=int(stats[2]))


def probe_fp32(op: int, iters: int, out, stream=None) -> int:
    """blink_probe_fp32 (include/blink_testing.h): launches the fp32 peak probe on `out` (cuda float32
    scratch), returns the flops of the launch; the caller times it."""
    lib = load_testing()
    flops = ctypes.c_int64(0)
    _check(lib.blink_probe_fp32(int(op), int(iters), out.data_ptr(), out.numel(), ctypes.byref(flops),
                                _stream_ptr(stream)), "blink_probe_fp32")
    return int(flops.value)


class Plan:
    """blink_plan_create / blink_plan_destroy and the calls that take a plan."""

    def __init__(self, ant_enu_m, freq_hz, n_pix: int, pixscale: float, weighting: int = NATURAL,
                 stream=None, options: "Options | dict | None" = None):
        lib = load()
        ant = np.ascontiguousarray(ant_enu_m, np.float64)
        fr = np.ascontiguousarray(freq_hz, np.float64).reshape(-1)
        if ant.ndim != 2 or ant.shape[1] != 3:
            raise ValueError("ant_enu_m must be [n_ant, 3]")
        self._h = ctypes.c_void_p(None)
        self._lib = lib
        if isinstance(options, dict):
            options = Options(**options)
        if options is None:
            _check(lib.blink_plan_create(ctypes.byref(self._h), ant.ctypes.data, ant.shape[0],
                                         fr.ctypes.data, fr.shape[0], int(n_pix), float(pixscale),
                                         int(weighting), _stream_ptr(stream)), "blink_plan_create")
        else:
            _check(lib.blink_plan_create_opts(ctypes.byref(self._h), ant.ctypes.data, ant.shape[0],
                                              fr.ctypes.data, fr.shape[0], int(n_pix), float(pixscale),
                                              int(weighting), _stream_ptr(stream), ctypes.byref(options)),
                   "blink_plan_create_opts")
        self._reserved_n_t = 0
        self._host_chunk_t = 0
        self.n_ant, self.n_ch, self.n_pix = ant.shape[0], fr.shape[0], int(n_pix)
        self.n_bl = self.query_i32(Q_N_BL)
        self.weighting = int(weighting)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.blink_plan_destroy(self._h)
            self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def refresh(self, ant_enu_m, stream=None):
        """blink_plan_refresh: new antenna coordinates, same everything else."""
        ant = np.ascontiguousarray(ant_enu_m, np.float64)
        if ant.shape != (self.n_ant, 3):
            raise ValueError("ant_enu_m must be [n_ant, 3]")
        _check(self._lib.blink_plan_refresh(self._h, ant.ctypes.data, _stream_ptr(stream)), "blink_plan_refresh")

    # ---- queries
    def _query(self, what, index, ctype, n=1):
        buf = (ctype * n)()
        _check(self._lib.blink_plan_query(self._h, what, index, ctypes.byref(buf)), "blink_plan_query")
        return buf[0] if n == 1 else list(buf)

    def query_i32(self, what, index=0):
        return int(self._query(what, index, ctypes.c_int32))

    def query_i64(self, what, index=0):
        return int(self._query(what, index, ctypes.c_int64))

    def n_dropped(self, ch):
        return self.query_i64(Q_N_DROPPED, ch)

    def wsum(self, ch):
        return self.query_i64(Q_WSUM, ch)

    def n_occ(self, ch):
        return self.query_i64(Q_N_OCC, ch)

    def bbox(self, ch):
        return tuple(self._query(Q_BBOX, ch, ctypes.c_int32, 2))

    def norm(self, ch):
        return float(self._query(Q_NORM, ch, ctypes.c_double))

    def _read(self, what, ch, n, dtype):
        out = np.empty(n, dtype)
        _check(self._lib.blink_plan_read(self._h, what, int(ch), out.ctypes.data, out.nbytes),
               "blink_plan_read")
        return out

    def cell_idx(self, ch):
        """int32 [n_bl] cell of V per baseline of channel ch (-1 dropped), host copy."""
        return self._read(Q_CELL_IDX, ch, self.n_bl, np.int32)

    def counts(self, ch):
        """uint32 [N, N] weight counts of channel ch, host copy."""
        return self._read(Q_COUNTS, ch, self.n_pix * self.n_pix, np.uint32).reshape(self.n_pix, self.n_pix)

    # ---- pre-gridding corrections (section 4.2)
    def set_corrections(self, gains=None, cable_len_m=None, l0: float = 0.0, m0: float = 0.0, stream=None):
        """blink_plan_set_corrections: gains complex [n_ch, n_ant] or None, cable lengths [n_ant] or None,
        new phase centre (l0, m0)."""
        g = c = None
        if gains is not None:
            g = np.ascontiguousarray(gains, np.complex128)
            if g.shape != (self.n_ch, self.n_ant):
                raise ValueError("gains must be [n_ch, n_ant]")
        if cable_len_m is not None:
            c = np.ascontiguousarray(cable_len_m, np.float64)
            if c.shape != (self.n_ant,):
                raise ValueError("cable_len_m must be [n_ant]")
        _check(self._lib.blink_plan_set_corrections(self._h, g.ctypes.data if g is not None else None,
                                                    c.ctypes.data if c is not None else None,
                                                    float(l0), float(m0), _stream_ptr(stream)),
               "blink_plan_set_corrections")

    def apply_corrections(self, on: bool, stream=None):
        """blink_plan_apply_corrections: on -> blink_grid / blink_grid_image multiply by the factors at load."""
        _check(self._lib.blink_plan_apply_corrections(self._h, 1 if on else 0, _stream_ptr(stream)),
               "blink_plan_apply_corrections")
        self._reserved_n_t = 0 if on else self._reserved_n_t     # the route, hence the scratch needed, may change

    def corr_table(self, ch):
        """complex64 [n_bl] correction factors of channel ch, host copy."""
        return self._read(Q_CORR, ch, self.n_bl, np.complex64)

    def correct(self, vis, out=None, stream=None):
        """blink_correct: out = vis * F (out may be vis itself)."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        assert tuple(vis.shape[1:]) == (self.n_ch, self.n_bl)
        if out is None:
            out = torch.empty_like(vis)
        assert out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous() and out.shape == vis.shape
        _check(self._lib.blink_correct(self._h, vis.data_ptr(), vis.shape[0], out.data_ptr(),
                                       _stream_ptr(stream)), "blink_correct")
        return out

    # ---- dynamic spectra (the stage after imaging)
    def dynspec(self, images, alpha: float, ref_state=None, out=None, stream=None):
        """blink_dynspec: images [n_t, n_ch, N, N] -> dynamic spectra [N, N, n_ch, n_t]; ref_state
        [n_ch, N, N] is updated in place (None: zero reference, no state kept)."""
        import torch
        n = self.n_pix
        assert images.is_cuda and images.dtype == torch.float32 and images.is_contiguous()
        assert tuple(images.shape[1:]) == (self.n_ch, n, n)
        n_t = images.shape[0]
        if ref_state is not None:
            assert ref_state.is_cuda and ref_state.dtype == torch.float32 and ref_state.is_contiguous()
            assert tuple(ref_state.shape) == (self.n_ch, n, n)
        if out is None:
            out = torch.empty((n, n, self.n_ch, n_t), dtype=torch.float32, device=images.device)
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
        assert tuple(out.shape) == (n, n, self.n_ch, n_t)
        _check(self._lib.blink_dynspec(self._h, images.data_ptr(), n_t, float(alpha),
                                       ref_state.data_ptr() if ref_state is not None else None,
                                       out.data_ptr(), _stream_ptr(stream)), "blink_dynspec")
        return out

    # ---- hot path
    def reserve(self, n_t: int):
        """blink_plan_reserve: the one place plan scratch is allocated (the hot calls never allocate and
        return BLINK_ERESERVE when it is too small)."""
        _check(self._lib.blink_plan_reserve(self._h, int(n_t)), "blink_plan_reserve")
        self._reserved_n_t = max(self._reserved_n_t, int(n_t))

    def _ensure_reserved(self, n_t: int, auto_reserve: bool):
        if auto_reserve and n_t > self._reserved_n_t:
            self.reserve(n_t)

    def validate(self, uv_grid, stream=None) -> int:
        """blink_grid_validate: number of cells of uv_grid that break blink_image's input contract."""
        import torch
        assert uv_grid.is_cuda and uv_grid.dtype == torch.complex64 and uv_grid.is_contiguous()
        assert tuple(uv_grid.shape[1:]) == (self.n_ch, self.n_pix, self.n_pix)
        n = ctypes.c_int64(0)
        _check(self._lib.blink_grid_validate(self._h, uv_grid.data_ptr(), uv_grid.shape[0], ctypes.byref(n),
                                             _stream_ptr(stream)), "blink_grid_validate")
        return int(n.value)

    def grid(self, vis, uv_grid=None, stream=None):
        """blink_grid: vis complex64 cuda [n_t, n_ch, n_bl] -> uv_grid complex64 [n_t, n_ch, N, N]."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        n_t = vis.shape[0]
        assert tuple(vis.shape[1:]) == (self.n_ch, self.n_bl)
        if uv_grid is None:
            uv_grid = torch.empty((n_t, self.n_ch, self.n_pix, self.n_pix), dtype=torch.complex64,
                                  device=vis.device)
        assert uv_grid.is_cuda and uv_grid.dtype == torch.complex64 and uv_grid.is_contiguous()
        assert tuple(uv_grid.shape) == (n_t, self.n_ch, self.n_pix, self.n_pix)
        _check(self._lib.blink_grid(self._h, vis.data_ptr(), n_t, uv_grid.data_ptr(),
                                    _stream_ptr(stream)), "blink_grid")
        return uv_grid

    def image(self, uv_grid, images=None, stream=None, auto_reserve=True):
        """blink_image: uv_grid complex64 [n_t, n_ch, N, N] -> images float32 [n_t, n_ch, N, N].
        auto_reserve: call blink_plan_reserve first when this n_t is larger than any reserved so far
        (a convenience of the binding; pass False to see the C call's own BLINK_ERESERVE)."""
        import torch
        assert uv_grid.is_cuda and uv_grid.dtype == torch.complex64 and uv_grid.is_contiguous()
        n_t = uv_grid.shape[0]
        assert tuple(uv_grid.shape[1:]) == (self.n_ch, self.n_pix, self.n_pix)
        if images is None:
            images = torch.empty((n_t, self.n_ch, self.n_pix, self.n_pix), dtype=torch.float32,
                                 device=uv_grid.device)
        assert images.is_cuda and images.dtype == torch.float32 and images.is_contiguous()
        self._ensure_reserved(n_t, auto_reserve)
        _check(self._lib.blink_image(self._h, uv_grid.data_ptr(), n_t, images.data_ptr(),
                                     _stream_ptr(stream)), "blink_image")
        return images

    def image_static(self, uv_grid, images, stream=None):
        """blink_image_static: blink_image for a caller that must not allocate device memory (a real-time
        loop that cannot take cudaMalloc's stall, a GPU whose memory is already spoken for).  The
        intermediate of the two passes lives in a 32 MiB array built into libblink.so instead of plan
        scratch, so no reserve() is needed and none is made; `images` is required because this wrapper
        does not allocate either.  BlinkError with status ECAPACITY when one snapshot's intermediate
        (8 N wu bytes) exceeds the array.  One array per GPU, shared by every plan: calls that overlap
        on the device corrupt each other, keep them on one stream."""
        import torch
        assert uv_grid.is_cuda and uv_grid.dtype == torch.complex64 and uv_grid.is_contiguous()
        n_t = uv_grid.shape[0]
        assert tuple(uv_grid.shape[1:]) == (self.n_ch, self.n_pix, self.n_pix)
        assert images.is_cuda and images.dtype == torch.float32 and images.is_contiguous()
        assert tuple(images.shape) == (n_t, self.n_ch, self.n_pix, self.n_pix)
        _check(self._lib.blink_image_static(self._h, uv_grid.data_ptr(), n_t, images.data_ptr(),
                                            _stream_ptr(stream)), "blink_image_static")
        return images

    def grid_image(self, vis, images=None, stream=None, auto_reserve=True):
        """blink_grid_image: vis complex64 [n_t, n_ch, n_bl] -> images float32 [n_t, n_ch, N, N]."""
        import torch
        assert vis.is_cuda and vis.dtype == torch.complex64 and vis.is_contiguous()
        n_t = vis.shape[0]
        assert tuple(vis.shape[1:]) == (self.n_ch, self.n_bl)
        if images is None:
            images = torch.empty((n_t, self.n_ch, self.n_pix, self.n_pix), dtype=torch.float32,
                                 device=vis.device)
        assert images.is_cuda and images.dtype == torch.float32 and images.is_contiguous()
        assert tuple(images.shape) == (n_t, self.n_ch, self.n_pix, self.n_pix)
        self._ensure_reserved(n_t, auto_reserve)
        _check(self._lib.blink_grid_image(self._h, vis.data_ptr(), n_t, images.data_ptr(),
                                          _stream_ptr(stream)), "blink_grid_image")
        return images

    def reserve_host(self, chunk_t: int):
        """blink_plan_reserve_host: staging of grid_image_host for chunks of chunk_t time steps (0: the plan
        picks the chunk, about 32 MiB each way)."""
        _check(self._lib.blink_plan_reserve_host(self._h, int(chunk_t)), "blink_plan_reserve_host")
        self._host_chunk_t = max(self._host_chunk_t, int(chunk_t), 1)
        self._reserved_n_t = max(self._reserved_n_t, int(chunk_t))

    def grid_image_host(self, vis_h, images_h, stream=None):
        """blink_grid_image_host: vis_h complex64 CPU tensor [n_t, n_ch, n_bl] (pinned for overlap) ->
        images_h float32 CPU tensor [n_t, n_ch, N, N]; asynchronous on the stream (synchronise it before
        reading images_h).  Without an earlier reserve_host the plan picks the chunk (reserve_host(0))."""
        import torch
        assert not vis_h.is_cuda and vis_h.dtype == torch.complex64 and vis_h.is_contiguous()
        n_t = vis_h.shape[0]
        assert tuple(vis_h.shape[1:]) == (self.n_ch, self.n_bl)
        assert not images_h.is_cuda and images_h.dtype == torch.float32 and images_h.is_contiguous()
        assert tuple(images_h.shape) == (n_t, self.n_ch, self.n_pix, self.n_pix)
        if self._host_chunk_t == 0:
            self.reserve_host(0)
        _check(self._lib.blink_grid_image_host(self._h, vis_h.data_ptr(), n_t, images_h.data_ptr(),
                                               _stream_ptr(stream)), "blink_grid_image_host")
        return images_h
