"""ctypes binding over libargus.so: argument marshalling only (every step of the path runs in the
CUDA kernels behind the C ABI of include/argus.h).  PyTorch supplies device memory and streams.

No CPU fallback exists: if the library cannot be loaded, every entry point raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

ARGUS_BILINEAR, ARGUS_LANCZOS3 = 0, 1
ARGUS_MASTERS_F32, ARGUS_MASTERS_F16 = 1, 2
ARGUS_OPT_PLAN_CACHE = 1
ARGUS_OPT_PROFILE = 2
ARGUS_OPT_FAST_PATH = 3
ARGUS_OPT_PLAN_OVERLAP = 4
ARGUS_OPT_SEGMENT_RASTER = 5
ARGUS_OPT_UNIT_MARGIN = 6
_KERNELS = {"bilinear": ARGUS_BILINEAR, "lanczos3": ARGUS_LANCZOS3, 0: 0, 1: 1}

EXPORTS = [
    "argus_strerror", "argus_version", "argus_ctx_create", "argus_ctx_destroy", "argus_ctx_set_option",
    "argus_last_cuda_error", "argus_launch_count", "argus_calibrate", "argus_prepare_masters", "argus_healpix_footprint", "argus_resample",
    "argus_coadd_accumulate", "argus_resample_coadd", "argus_plan_info", "argus_profile_read",
    "argus_resample_host", "argus_resample_coadd_host", "argus_reduce_frame_host", "argus_host_wait", "argus_subtract_tiles", "argus_segment_products", "argus_background_map", "argus_detect_sources",
    "argus_background_map_static", "argus_detect_frame", "argus_detect_frame_info",
]


class ArgusError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        msg = "%s failed: %s (%d)" % (where, _strerror(status), status)
        super().__init__(msg + (" " + detail if detail else ""))


class _Wcs(C.Structure):
    _fields_ = [("crval", C.c_double * 2), ("crpix", C.c_double * 2), ("cd", (C.c_double * 2) * 2),
                ("sip_order", C.c_int32), ("reserved", C.c_int32), ("ap", C.c_double * 36), ("bp", C.c_double * 36)]


class _Frame(C.Structure):
    _fields_ = [("raw", C.c_void_p), ("bias", C.c_void_p), ("dark", C.c_void_p), ("flat", C.c_void_p),
                ("bpm", C.c_void_p), ("t_exp", C.c_float), ("sat_adu", C.c_int32), ("flat_min", C.c_float),
                ("cal", C.c_void_p), ("mask", C.c_void_p), ("offset", C.c_void_p), ("gain", C.c_void_p),
                ("masters_format", C.c_int32), ("reserved", C.c_int32)]


class _Coadd(C.Structure):
    _fields_ = [("tiles", C.c_void_p), ("n_tiles", C.c_int64), ("nside_tile", C.c_int64)]


class _SubParams(C.Structure):
    _fields_ = [("match", C.c_int32), ("n_min", C.c_int32), ("sci_wmin", C.c_float), ("ref_wmin", C.c_float),
                ("read_noise", C.c_float), ("gain", C.c_float), ("k_sigma", C.c_float), ("reserved", C.c_float)]


class _PlanStats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_footprint", "n_tiles", "n_inside", "n_border", "n_exact", "n_empty", "n_units", "n_stray")]


_lib = None


def library_path() -> str:
    """libargus.so beside this file; ARGUS_LIBRARY names another build of the same sources (the ARGUS_DEBUG_BOUNDS build of
    tests/test_gpu_debug_bounds.py)."""
    return os.environ.get("ARGUS_LIBRARY") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "libargus.so")


def load_library():
    """Load libargus.so (built in-tree by ``_build.build()``).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    # rebuild in-tree when the sources are newer than the library (needs nvcc; never falls back to CPU).  A failed rebuild
    # of stale sources is an error: running an old library against new sources would hide it.  Without nvcc (a box that
    # only received the built .so) the existing library is used as it is.
    from . import _build
    if not os.environ.get("ARGUS_LIBRARY"):
        try:
            _build.build()
        except FileNotFoundError:
            if not os.path.exists(path):
                raise
    if not os.path.exists(path):
        raise ImportError("libargus.so not built: run `python -m paper_2207_14304_b200._build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    L = C.CDLL(path)
    vp, i64, i32, f32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_size_t
    L.argus_strerror.restype = C.c_char_p
    L.argus_strerror.argtypes = [C.c_int]
    L.argus_version.restype = C.c_int
    L.argus_ctx_create.argtypes = [C.POINTER(vp), C.c_int, i64]
    L.argus_ctx_destroy.argtypes = [vp]
    L.argus_ctx_set_option.argtypes = [vp, C.c_int, i64]
    L.argus_last_cuda_error.argtypes = [vp]
    L.argus_launch_count.argtypes = [vp]
    L.argus_launch_count.restype = i64
    L.argus_calibrate.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, f32, i32, f32, vp, vp, vp]
    L.argus_prepare_masters.argtypes = [vp, vp, vp, vp, vp, i64, i64, f32, f32, C.c_int, vp, vp, vp]
    L.argus_healpix_footprint.argtypes = [vp, C.POINTER(_Wcs), i64, i64, i64, vp, sz, C.POINTER(sz), vp]
    L.argus_resample.argtypes = [vp, C.POINTER(_Frame), C.POINTER(_Wcs), i64, i64, i64, C.c_int, f32, vp, sz, vp, vp, vp]
    L.argus_coadd_accumulate.argtypes = [vp, C.POINTER(_Coadd), i64, vp, vp, vp, vp, vp, sz, vp, vp]
    L.argus_resample_coadd.argtypes = [vp, C.POINTER(_Frame), C.POINTER(_Wcs), i64, i64, i64, C.c_int, f32,
                                       C.POINTER(_Coadd), vp, vp, vp, vp]
    L.argus_resample_host.argtypes = [vp, C.POINTER(_Frame), C.POINTER(_Wcs), i64, i64, i64, C.c_int, f32, sz, vp, vp, vp]
    L.argus_resample_coadd_host.argtypes = [vp, C.POINTER(_Frame), C.POINTER(_Wcs), i64, i64, i64, C.c_int, f32,
                                            C.POINTER(_Coadd), vp, vp, vp, vp]
    L.argus_reduce_frame_host.argtypes = [vp, C.POINTER(_Frame), C.POINTER(_Wcs), i64, i64, i64, C.c_int, f32, i64, sz, sz, vp, vp, vp,
                                          vp, vp, vp]
    L.argus_host_wait.argtypes = [vp]
    L.argus_segment_products.argtypes = [vp, i64, i64, vp, vp, vp, sz, vp, sz, C.POINTER(_Coadd), vp, vp, vp, vp, vp, sz,
                                         vp, C.POINTER(sz), vp]
    L.argus_background_map.argtypes = [vp, C.POINTER(_Frame), i64, i64, i32, i32, vp, vp, vp, vp, vp, vp]
    L.argus_detect_sources.argtypes = [vp, C.POINTER(_Frame), i64, i64, i32, vp, vp, f32, vp, sz, vp, C.POINTER(sz), vp]
    L.argus_detect_frame.argtypes = [vp, C.POINTER(_Frame), i64, i64, i32, i32, f32, vp, vp, vp, sz, vp, C.POINTER(sz), vp]
    L.argus_detect_frame_info.argtypes = [vp, C.POINTER(i64), vp]
    L.argus_background_map_static.argtypes = [C.POINTER(_Frame), i64, i64, i32, i32, vp, vp, C.POINTER(i32), vp]
    L.argus_subtract_tiles.argtypes = [vp, C.POINTER(_Coadd), i64, vp, vp, vp, vp, C.POINTER(_SubParams), vp, vp, vp, vp, vp, vp, sz,
                                       vp, C.POINTER(sz), vp]
    L.argus_plan_info.argtypes = [vp, C.POINTER(_PlanStats), vp]
    L.argus_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(i64), vp]
    _lib = L
    return L


def _strerror(status: int) -> str:
    try:
        return load_library().argus_strerror(int(status)).decode()
    except Exception:  # pragma: no cover
        return "status %d" % status


def _wcs_struct(w) -> _Wcs:
    """Accepts synth.Wcs-like objects (crval, crpix, cd, sip_order, ap, bp) or a flat float64[81] array."""
    s = _Wcs()
    if hasattr(w, "crval"):
        crval, crpix, cd, order, ap, bp = w.crval, w.crpix, w.cd, w.sip_order, w.ap, w.bp
    else:
        a = [float(v) for v in w]
        crval, crpix, cd = a[0:2], a[2:4], ((a[4], a[5]), (a[6], a[7]))
        order, ap, bp = int(a[8]), a[9:45], a[45:81]
    s.crval[0], s.crval[1] = float(crval[0]), float(crval[1])
    s.crpix[0], s.crpix[1] = float(crpix[0]), float(crpix[1])
    for i in range(2):
        for j in range(2):
            s.cd[i][j] = float(cd[i][j])
    s.sip_order = int(order)
    for i in range(36):
        s.ap[i] = float(ap[i])
        s.bp[i] = float(bp[i])
    return s


def _dev(t, dtype, name, allow_none=False):
    if t is None:
        if allow_none:
            return None
        raise ValueError("%s is required" % name)
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor" % name)
    if t.dtype != dtype:
        raise TypeError("%s must have dtype %s, got %s" % (name, dtype, t.dtype))
    if not t.is_contiguous():
        raise ValueError("%s must be contiguous" % name)
    return t.data_ptr()


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _frame_struct(raw=None, bias=None, dark=None, flat=None, bpm=None, t_exp=0.0, sat_adu=65535, flat_min=0.1,
                  cal=None, mask=None, offset=None, gain=None) -> _Frame:
    f = _Frame()
    if raw is not None and offset is not None:      # pre-fused masters (argus_prepare_masters): float32 or float16 tensors
        if offset.dtype != gain.dtype or offset.dtype not in (torch.float32, torch.float16):
            raise TypeError("offset and gain must both be float32 or both float16")
        f.raw = _dev(raw, torch.uint16, "raw")
        f.offset = _dev(offset, offset.dtype, "offset")
        f.gain = _dev(gain, gain.dtype, "gain")
        f.masters_format = ARGUS_MASTERS_F32 if offset.dtype == torch.float32 else ARGUS_MASTERS_F16
        if offset.shape != raw.shape or gain.shape != raw.shape:
            raise ValueError("masters must have the frame's shape")
    elif raw is not None:
        f.raw = _dev(raw, torch.uint16, "raw")
        f.bias = _dev(bias, torch.float32, "bias")
        f.dark = _dev(dark, torch.float32, "dark")
        f.flat = _dev(flat, torch.float32, "flat")
        f.bpm = _dev(bpm, torch.uint8, "bpm", allow_none=True)
        for t in (bias, dark, flat) + ((bpm,) if bpm is not None else ()):
            if t.shape != raw.shape:
                raise ValueError("masters must have the frame's shape")
    else:
        f.cal = _dev(cal, torch.float32, "cal")
        f.mask = _dev(mask, torch.uint8, "mask")
        if cal.shape != mask.shape:
            raise ValueError("cal and mask must have the same shape")
    f.t_exp, f.sat_adu, f.flat_min = float(t_exp), int(sat_adu), float(flat_min)
    return f


class Context:
    """argus_ctx handle: owns the plan scratch on one device."""

    def __init__(self, device: int | None = None, max_tiles: int = 0):
        L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("CUDA device required: the argus hot path has no CPU fallback")
        self.device = torch.cuda.current_device() if device is None else int(device)
        h = C.c_void_p()
        rc = L.argus_ctx_create(C.byref(h), self.device, int(max_tiles))
        if rc:
            raise ArgusError(rc, "argus_ctx_create")
        self._h = h

    def set_plan_cache(self, on: bool):
        rc = load_library().argus_ctx_set_option(self._h, ARGUS_OPT_PLAN_CACHE, 1 if on else 0)
        if rc:
            raise ArgusError(rc, "argus_ctx_set_option")

    def set_profile(self, on: bool):
        rc = load_library().argus_ctx_set_option(self._h, ARGUS_OPT_PROFILE, 1 if on else 0)
        if rc:
            raise ArgusError(rc, "argus_ctx_set_option")

    def set_fast_path(self, on):
        """False / 0: general kernel only; True / 1: default choice; 2: tile kernel only; 3: unit kernel where possible;
        4: default choice without the two-stage Lanczos-3 form of fine grids (include/argus.h, ARGUS_OPT_FAST_PATH)."""
        rc = load_library().argus_ctx_set_option(self._h, ARGUS_OPT_FAST_PATH, int(on))
        if rc:
            raise ArgusError(rc, "argus_ctx_set_option")

    def set_plan_overlap(self, on: bool):
        rc = load_library().argus_ctx_set_option(self._h, ARGUS_OPT_PLAN_OVERLAP, 1 if on else 0)
        if rc:
            raise ArgusError(rc, "argus_ctx_set_option")

    def set_unit_margin(self, delta: int):
        rc = load_library().argus_ctx_set_option(self._h, ARGUS_OPT_UNIT_MARGIN, int(delta))
        if rc:
            raise ArgusError(rc, "argus_ctx_set_option")

    def set_segment_raster(self, on: bool):
        rc = load_library().argus_ctx_set_option(self._h, ARGUS_OPT_SEGMENT_RASTER, 1 if on else 0)
        if rc:
            raise ArgusError(rc, "argus_ctx_set_option")

    def launch_count(self) -> int:
        return int(load_library().argus_launch_count(self._h))

    def profile_read(self, stream=None):
        """Returns (plan_ms_total, kernel_ms_total, n_calls) of the calls recorded since profiling was enabled."""
        p, k, n = C.c_double(), C.c_double(), C.c_int64()
        rc = load_library().argus_profile_read(self._h, C.byref(p), C.byref(k), C.byref(n), _stream(stream))
        if rc:
            raise ArgusError(rc, "argus_profile_read")
        return p.value, k.value, int(n.value)

    def last_cuda_error(self) -> int:
        return int(load_library().argus_last_cuda_error(self._h))

    def close(self):
        if getattr(self, "_h", None):
            load_library().argus_ctx_destroy(self._h)
            self._h = None

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass


def _check(ctx, rc, where):
    if rc:
        detail = ""
        if rc == -8:
            detail = "cudaError=%d" % ctx.last_cuda_error()
        raise ArgusError(rc, where, detail)


def argus_calibrate(ctx, raw, bias, dark, flat, bpm, t_exp, sat_adu=65535, flat_min=0.1, cal_out=None, mask_out=None,
                    stream=None):
    """A2 standalone.  Returns (cal float32 [H][W], mask uint8 [H][W])."""
    H, W = raw.shape
    if cal_out is None:
        cal_out = torch.empty((H, W), dtype=torch.float32, device=raw.device)
    if mask_out is None:
        mask_out = torch.empty((H, W), dtype=torch.uint8, device=raw.device)
    f = _frame_struct(raw, bias, dark, flat, bpm, t_exp, sat_adu, flat_min)
    rc = load_library().argus_calibrate(ctx._h, f.raw, f.bias, f.dark, f.flat, f.bpm, W, H, float(t_exp), int(sat_adu),
                                        float(flat_min), _dev(cal_out, torch.float32, "cal_out"),
                                        _dev(mask_out, torch.uint8, "mask_out"), _stream(stream))
    _check(ctx, rc, "argus_calibrate")
    return cal_out, mask_out


def argus_prepare_masters(ctx, bias, dark, flat, bpm, t_exp, flat_min=0.1, dtype=torch.float32, offset_out=None,
                          gain_out=None, stream=None):
    """offset = bias + dark * t_exp and gain = 1 / flat (NaN = invalid) as float32 or float16 CUDA
    tensors, once per pointing.  Returns (offset, gain): pass them as offset= / gain= instead of bias= / dark= / flat=."""
    if dtype not in (torch.float32, torch.float16):
        raise TypeError("dtype must be torch.float32 or torch.float16")
    H, W = bias.shape
    if offset_out is None:
        offset_out = torch.empty((H, W), dtype=dtype, device=bias.device)
    if gain_out is None:
        gain_out = torch.empty((H, W), dtype=dtype, device=bias.device)
    rc = load_library().argus_prepare_masters(
        ctx._h, _dev(bias, torch.float32, "bias"), _dev(dark, torch.float32, "dark"), _dev(flat, torch.float32, "flat"),
        _dev(bpm, torch.uint8, "bpm", allow_none=True), W, H, float(t_exp), float(flat_min),
        ARGUS_MASTERS_F32 if dtype == torch.float32 else ARGUS_MASTERS_F16, _dev(offset_out, dtype, "offset_out"),
        _dev(gain_out, dtype, "gain_out"), _stream(stream))
    _check(ctx, rc, "argus_prepare_masters")
    return offset_out, gain_out


def argus_healpix_footprint(ctx, wcs, W, H, nside, idx_out=None, want_indices=True, stream=None):
    """A0 + A1.  Returns (n, idx) with idx an ascending int64 CUDA tensor (None if want_indices is False)."""
    L = load_library()
    w = _wcs_struct(wcs)
    n = C.c_size_t(0)
    if idx_out is None:
        rc = L.argus_healpix_footprint(ctx._h, C.byref(w), W, H, nside, None, 0, C.byref(n), _stream(stream))
        _check(ctx, rc, "argus_healpix_footprint")
        if not want_indices:
            return int(n.value), None
        idx_out = torch.empty(int(n.value), dtype=torch.int64, device="cuda:%d" % ctx.device)
    rc = L.argus_healpix_footprint(ctx._h, C.byref(w), W, H, nside, _dev(idx_out, torch.int64, "idx_out"),
                                   idx_out.numel(), C.byref(n), _stream(stream))
    _check(ctx, rc, "argus_healpix_footprint")
    return int(n.value), idx_out[: int(n.value)]


def argus_resample(ctx, wcs, W, H, nside, kernel, value_out, weight_out, idx=None, w_min=0.5, stream=None, **frame):
    """A3-A5 (+A2 fused when raw/bias/dark/flat are given, else cal/mask).  Asynchronous."""
    f = _frame_struct(**frame)
    w = _wcs_struct(wcs)
    n = idx.numel() if idx is not None else min(value_out.numel(), weight_out.numel())
    if idx is not None and (value_out.numel() < n or weight_out.numel() < n):
        raise ValueError("outputs smaller than idx")
    rc = load_library().argus_resample(ctx._h, C.byref(f), C.byref(w), W, H, nside, _KERNELS[kernel], float(w_min),
                                       _dev(idx, torch.int64, "idx", allow_none=True), n,
                                       _dev(value_out, torch.float32, "value_out"),
                                       _dev(weight_out, torch.float32, "weight_out"), _stream(stream))
    _check(ctx, rc, "argus_resample")


def _host_frame_struct(raw_host, bias, dark, flat, offset, gain, t_exp, sat_adu, flat_min) -> _Frame:
    """argus_frame with a HOST raw pointer and DEVICE masters (bias / dark / flat, or the pre-fused offset / gain)."""
    f = _Frame()
    f.raw = raw_host.data_ptr()
    if offset is not None:
        if offset.dtype != gain.dtype or offset.dtype not in (torch.float32, torch.float16):
            raise TypeError("offset and gain must both be float32 or both float16")
        f.offset = _dev(offset, offset.dtype, "offset")
        f.gain = _dev(gain, gain.dtype, "gain")
        f.masters_format = ARGUS_MASTERS_F32 if offset.dtype == torch.float32 else ARGUS_MASTERS_F16
    else:
        f.bias = _dev(bias, torch.float32, "bias")
        f.dark = _dev(dark, torch.float32, "dark")
        f.flat = _dev(flat, torch.float32, "flat")
    f.t_exp, f.sat_adu, f.flat_min = float(t_exp), int(sat_adu), float(flat_min)
    return f


def argus_resample_host(ctx, wcs, W, H, nside, kernel, n, raw_host, value_host, weight_host, w_min=0.5, stream=None,
                        bias=None, dark=None, flat=None, t_exp=0.0, sat_adu=65535, flat_min=0.1, offset=None, gain=None):
    """A2-A5 with HOST frame / outputs (CPU tensors, pinned for asynchronous copies); masters are CUDA tensors.
    Asynchronous: call argus_host_wait(ctx) before reading value_host / weight_host."""
    for t, dt, name in ((raw_host, torch.uint16, "raw_host"), (value_host, torch.float32, "value_host"),
                        (weight_host, torch.float32, "weight_host")):
        if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != dt or not t.is_contiguous():
            raise TypeError("%s must be a contiguous CPU tensor of dtype %s" % (name, dt))
    if raw_host.numel() != W * H or value_host.numel() < n or weight_host.numel() < n:
        raise ValueError("host buffers too small")
    f = _host_frame_struct(raw_host, bias, dark, flat, offset, gain, t_exp, sat_adu, flat_min)
    w = _wcs_struct(wcs)
    rc = load_library().argus_resample_host(ctx._h, C.byref(f), C.byref(w), W, H, nside, _KERNELS[kernel], float(w_min), int(n),
                                            value_host.data_ptr(), weight_host.data_ptr(), _stream(stream))
    _check(ctx, rc, "argus_resample_host")


def argus_reduce_frame_host(ctx, wcs, W, H, nside, kernel, n, raw_host, seg16_host, mini_id_host, mini_value_host,
                            mini_weight_host, n_mini_host, nside_mini=1 << 14, w_min=0.5, stream=None, bias=None, dark=None,
                            flat=None, t_exp=0.0, sat_adu=65535, flat_min=0.1, offset=None, gain=None):
    """The per-frame product with HOST buffers (pinned CPU tensors): binary16 segment data (int16 / uint16 / float16 tensor
    of n elements) + low-resolution map (mini_* of one capacity, n_mini_host int64[1]).  Masters are CUDA tensors."""
    cap = mini_id_host.numel()
    for t, dts, name in ((raw_host, (torch.uint16,), "raw_host"), (seg16_host, (torch.int16, torch.uint16, torch.float16), "seg16_host"),
                         (mini_id_host, (torch.int64,), "mini_id_host"), (mini_value_host, (torch.float32,), "mini_value_host"),
                         (mini_weight_host, (torch.float32,), "mini_weight_host"), (n_mini_host, (torch.int64,), "n_mini_host")):
        if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype not in dts or not t.is_contiguous():
            raise TypeError("%s must be a contiguous CPU tensor of dtype %s" % (name, dts))
    if raw_host.numel() != W * H or seg16_host.numel() < n or mini_value_host.numel() < cap or mini_weight_host.numel() < cap:
        raise ValueError("host buffers too small")
    f = _host_frame_struct(raw_host, bias, dark, flat, offset, gain, t_exp, sat_adu, flat_min)
    w = _wcs_struct(wcs)
    rc = load_library().argus_reduce_frame_host(ctx._h, C.byref(f), C.byref(w), W, H, nside, _KERNELS[kernel], float(w_min),
                                                int(nside_mini), int(n), int(cap), seg16_host.data_ptr(), mini_id_host.data_ptr(),
                                                mini_value_host.data_ptr(), mini_weight_host.data_ptr(), n_mini_host.data_ptr(),
                                                _stream(stream))
    _check(ctx, rc, "argus_reduce_frame_host")


def argus_host_wait(ctx):
    _check(ctx, load_library().argus_host_wait(ctx._h), "argus_host_wait")


def _coadd_struct(tiles, nside_tile) -> _Coadd:
    c = _Coadd()
    c.tiles = _dev(tiles, torch.int64, "tiles")
    c.n_tiles = tiles.numel()
    c.nside_tile = int(nside_tile)
    return c


def argus_coadd_accumulate(ctx, tiles, nside_tile, nside, sum_, wsum, idx, value, weight, n_skipped=None, stream=None):
    """A6 on an explicit (idx, value, weight) list.  Asynchronous."""
    lay = _coadd_struct(tiles, nside_tile)
    rc = load_library().argus_coadd_accumulate(ctx._h, C.byref(lay), nside, _dev(sum_, torch.float32, "sum"),
                                               _dev(wsum, torch.float32, "wsum"), _dev(idx, torch.int64, "idx"),
                                               _dev(value, torch.float32, "value"), _dev(weight, torch.float32, "weight"),
                                               idx.numel(), _dev(n_skipped, torch.int64, "n_skipped", allow_none=True),
                                               _stream(stream))
    _check(ctx, rc, "argus_coadd_accumulate")


def argus_resample_coadd(ctx, wcs, W, H, nside, kernel, tiles, nside_tile, sum_, wsum, n_skipped=None, w_min=0.5,
                         stream=None, **frame):
    """A2-A6 fused.  Asynchronous."""
    f = _frame_struct(**frame)
    w = _wcs_struct(wcs)
    lay = _coadd_struct(tiles, nside_tile)
    rc = load_library().argus_resample_coadd(ctx._h, C.byref(f), C.byref(w), W, H, nside, _KERNELS[kernel], float(w_min),
                                             C.byref(lay), _dev(sum_, torch.float32, "sum"),
                                             _dev(wsum, torch.float32, "wsum"),
                                             _dev(n_skipped, torch.int64, "n_skipped", allow_none=True), _stream(stream))
    _check(ctx, rc, "argus_resample_coadd")


def argus_resample_coadd_host(ctx, wcs, W, H, nside, kernel, raw_host, tiles, nside_tile, sum_, wsum, n_skipped=None,
                              w_min=0.5, stream=None, bias=None, dark=None, flat=None, t_exp=0.0, sat_adu=65535, flat_min=0.1,
                              offset=None, gain=None):
    """A2-A6 fused with the raw frame in HOST memory (pinned CPU tensor); masters and the coadd are CUDA tensors."""
    if not isinstance(raw_host, torch.Tensor) or raw_host.is_cuda or raw_host.dtype != torch.uint16 or not raw_host.is_contiguous():
        raise TypeError("raw_host must be a contiguous CPU uint16 tensor")
    if raw_host.numel() != W * H:
        raise ValueError("raw_host does not hold W * H pixels")
    f = _host_frame_struct(raw_host, bias, dark, flat, offset, gain, t_exp, sat_adu, flat_min)
    w = _wcs_struct(wcs)
    lay = _coadd_struct(tiles, nside_tile)
    rc = load_library().argus_resample_coadd_host(ctx._h, C.byref(f), C.byref(w), W, H, nside, _KERNELS[kernel], float(w_min),
                                                  C.byref(lay), _dev(sum_, torch.float32, "sum"),
                                                  _dev(wsum, torch.float32, "wsum"),
                                                  _dev(n_skipped, torch.int64, "n_skipped", allow_none=True), _stream(stream))
    _check(ctx, rc, "argus_resample_coadd_host")


def argus_segment_products(ctx, nside, nside_mini, idx, value, weight, targets, seg16=None, mini_id=None, mini_value=None,
                           mini_weight=None, mini_keep=None, tiles=None, nside_tile=None, n_mini_dev=None, sync=True,
                           stream=None):
    """Segment products on caller-allocated CUDA tensors; seg16 is an int16/uint16 tensor that
    receives binary16 bit patterns.  Returns n_mini when sync, else None.  Capacity = mini_id.numel()."""
    cap = 0 if mini_id is None else mini_id.numel()
    for name, t, dt in (("mini_value", mini_value, torch.float32), ("mini_weight", mini_weight, torch.float32),
                        ("mini_keep", mini_keep, torch.uint8)):
        if t is not None and t.numel() < cap:
            raise ValueError("%s is shorter than mini_id" % name)
    lay = _coadd_struct(tiles, nside_tile) if tiles is not None else None
    n = idx.numel()
    if value.numel() != n or weight.numel() != n:
        raise ValueError("idx, value and weight differ in length")
    if seg16 is not None:
        if seg16.dtype not in (torch.int16, torch.uint16, torch.float16):
            raise TypeError("seg16 must be a 16-bit tensor")
        need = n if tiles is None else tiles.numel() * (nside // int(nside_tile)) ** 2
        if seg16.numel() < need:
            raise ValueError("seg16 holds %d elements, %d needed" % (seg16.numel(), need))
    nm = C.c_size_t(0)
    rc = load_library().argus_segment_products(
        ctx._h, int(nside), int(nside_mini), _dev(idx, torch.int64, "idx") if n else None,
        _dev(value, torch.float32, "value") if n else None, _dev(weight, torch.float32, "weight") if n else None, n,
        _dev(targets, torch.int64, "targets") if targets is not None and targets.numel() else None,
        0 if targets is None else targets.numel(), C.byref(lay) if lay is not None else None,
        _dev(seg16, seg16.dtype, "seg16") if seg16 is not None else None,
        _dev(mini_id, torch.int64, "mini_id", allow_none=True), _dev(mini_value, torch.float32, "mini_value", allow_none=True),
        _dev(mini_weight, torch.float32, "mini_weight", allow_none=True),
        _dev(mini_keep, torch.uint8, "mini_keep", allow_none=True), cap,
        _dev(n_mini_dev, torch.int64, "n_mini_dev", allow_none=True), C.byref(nm) if sync else None, _stream(stream))
    if rc == -6 and sync:
        raise ArgusError(rc, "argus_segment_products", "n_mini=%d" % nm.value)
    _check(ctx, rc, "argus_segment_products")
    return int(nm.value) if sync else None


# numpy view of argus_source records (argus.h)
SOURCE_DTYPE = [("x", "<i4"), ("y", "<i4"), ("peak", "<f4"), ("flux", "<f4"), ("cx", "<f4"), ("cy", "<f4"), ("bkg", "<f4"),
                ("nse", "<f4")]


def argus_background_map(ctx, W, H, bkg_out, nse_out, cell=64, n_min=16, med_out=None, sig_out=None, ngood_out=None,
                         stream=None, **frame):
    """Median-filtered background and noise grids into caller-allocated float32 CUDA tensors of
    ceil(H / cell) * ceil(W / cell) elements.  frame: raw= bias= dark= flat= [bpm=] t_exp= ... or cal= mask=."""
    g = -(-int(H) // int(cell)) * -(-int(W) // int(cell))
    for name, t in (("bkg_out", bkg_out), ("nse_out", nse_out), ("med_out", med_out), ("sig_out", sig_out),
                    ("ngood_out", ngood_out)):
        if t is not None and t.numel() < g:
            raise ValueError("%s holds %d elements, %d needed" % (name, t.numel(), g))
    f = _frame_struct(**frame)
    rc = load_library().argus_background_map(
        ctx._h, C.byref(f), int(W), int(H), int(cell), int(n_min), _dev(bkg_out, torch.float32, "bkg_out"),
        _dev(nse_out, torch.float32, "nse_out"), _dev(med_out, torch.float32, "med_out", allow_none=True),
        _dev(sig_out, torch.float32, "sig_out", allow_none=True), _dev(ngood_out, torch.int32, "ngood_out", allow_none=True),
        _stream(stream))
    _check(ctx, rc, "argus_background_map")


ARGUS_BG_STATIC_MAX_CELLS = 1 << 20


def argus_background_map_static(W, H, bkg_out, nse_out, cell=64, n_min=16, stream=None, **frame):
    """argus_background_map without a context and without any allocation: the cell scratch is a file-scope device array of
    the library holding ARGUS_BG_STATIC_MAX_CELLS cells (more: ARGUS_ERR_CAPACITY).  Runs on the tensors' device, which
    must be the current one; calls sharing a device must not overlap on the GPU."""
    g = -(-int(H) // int(cell)) * -(-int(W) // int(cell))
    for name, t in (("bkg_out", bkg_out), ("nse_out", nse_out)):
        if t.numel() < g:
            raise ValueError("%s holds %d elements, %d needed" % (name, t.numel(), g))
    if bkg_out.device.index != torch.cuda.current_device():
        raise ValueError("argus_background_map_static works on the current device")
    f = _frame_struct(**frame)
    err = C.c_int32(0)
    rc = load_library().argus_background_map_static(
        C.byref(f), int(W), int(H), int(cell), int(n_min), _dev(bkg_out, torch.float32, "bkg_out"),
        _dev(nse_out, torch.float32, "nse_out"), C.byref(err), _stream(stream))
    if rc:
        detail = ""
        if rc == -8:
            detail = "cudaError=%d" % err.value
        elif rc == -6:
            detail = "%d cells > ARGUS_BG_STATIC_MAX_CELLS = %d" % (g, ARGUS_BG_STATIC_MAX_CELLS)
        raise ArgusError(rc, "argus_background_map_static", detail)


def argus_detect_sources(ctx, W, H, bkg, nse, out, cell=64, k_sigma=5.0, n_dev=None, sync=True, stream=None, **frame):
    """Source detection.  out: uint8 CUDA tensor of 32 * capacity bytes (argus_source records, view the
    host copy with SOURCE_DTYPE) or None to count.  Returns the number of sources found when sync, else None."""
    cap = 0 if out is None else out.numel() // 32
    if out is not None and out.dtype != torch.uint8:
        raise TypeError("out must be a uint8 tensor (32 bytes per record)")
    g = -(-int(H) // int(cell)) * -(-int(W) // int(cell))
    if bkg.numel() < g or nse.numel() < g:
        raise ValueError("bkg / nse hold fewer than %d cells" % g)
    f = _frame_struct(**frame)
    n = C.c_size_t(0)
    rc = load_library().argus_detect_sources(
        ctx._h, C.byref(f), int(W), int(H), int(cell), _dev(bkg, torch.float32, "bkg"), _dev(nse, torch.float32, "nse"),
        float(k_sigma), _dev(out, torch.uint8, "out", allow_none=True), cap, _dev(n_dev, torch.int64, "n_dev", allow_none=True),
        C.byref(n) if sync else None, _stream(stream))
    if rc == -6 and sync:
        raise ArgusError(rc, "argus_detect_sources", "n_sources=%d" % n.value)
    _check(ctx, rc, "argus_detect_sources")
    return int(n.value) if sync else None


def argus_detect_frame(ctx, W, H, bkg_out, nse_out, out, cell=64, n_min=16, k_sigma=5.0, n_dev=None, sync=True, stream=None,
                       **frame):
    """argus_background_map + argus_detect_sources in one call that reads the frame once (identical results).  Returns the
    number of sources found when sync, else None."""
    cap = 0 if out is None else out.numel() // 32
    if out is not None and out.dtype != torch.uint8:
        raise TypeError("out must be a uint8 tensor (32 bytes per record)")
    g = -(-int(H) // int(cell)) * -(-int(W) // int(cell))
    if bkg_out.numel() < g or nse_out.numel() < g:
        raise ValueError("bkg_out / nse_out hold fewer than %d cells" % g)
    f = _frame_struct(**frame)
    n = C.c_size_t(0)
    rc = load_library().argus_detect_frame(
        ctx._h, C.byref(f), int(W), int(H), int(cell), int(n_min), float(k_sigma), _dev(bkg_out, torch.float32, "bkg_out"),
        _dev(nse_out, torch.float32, "nse_out"), _dev(out, torch.uint8, "out", allow_none=True), cap,
        _dev(n_dev, torch.int64, "n_dev", allow_none=True), C.byref(n) if sync else None, _stream(stream))
    if rc == -6 and sync:
        raise ArgusError(rc, "argus_detect_frame", "n_sources=%d" % n.value)
    _check(ctx, rc, "argus_detect_frame")
    return int(n.value) if sync else None


def argus_detect_frame_info(ctx, stream=None) -> int:
    """Tiles the last argus_detect_frame scanned in full (synchronises)."""
    v = C.c_int64(0)
    rc = load_library().argus_detect_frame_info(ctx._h, C.byref(v), _stream(stream))
    _check(ctx, rc, "argus_detect_frame_info")
    return int(v.value)


# numpy view of argus_transient records (argus.h)
TRANSIENT_DTYPE = [("pixel", "<i8"), ("sig", "<f4"), ("diff", "<f4"), ("flux", "<f4"), ("noise", "<f4"), ("tile_rank", "<i4"),
                   ("reserved", "<i4")]
_MATCH = {"none": 0, "affine": 1, 0: 0, 1: 1}


def argus_subtract_tiles(ctx, tiles, nside_tile, nside, sci_sum, sci_wsum, ref_sum, ref_wsum, diff_out, sig_out=None, out=None,
                         match="affine", n_min=16, sci_wmin=0.5, ref_wmin=0.5, read_noise=1.7, gain=1.0, k_sigma=5.0,
                         alpha_out=None, beta_out=None, nvalid_out=None, n_dev=None, sync=True, stream=None):
    """Direct image subtraction per tile on the tile-dense (sum, wsum) pairs of a science frame and a
    reference coadd.  out: uint8 CUDA tensor of 32 * capacity bytes (argus_transient records, view the host copy with
    TRANSIENT_DTYPE) or None to count.  Returns the number of candidates when sync, else None."""
    lay = _coadd_struct(tiles, nside_tile)
    n_slots = tiles.numel() * (int(nside) // int(nside_tile)) ** 2
    for name, t in (("sci_sum", sci_sum), ("sci_wsum", sci_wsum), ("ref_sum", ref_sum), ("ref_wsum", ref_wsum),
                    ("diff_out", diff_out), ("sig_out", sig_out)):
        if t is not None and t.numel() < n_slots:
            raise ValueError("%s holds %d elements, %d needed" % (name, t.numel(), n_slots))
    for name, t in (("alpha_out", alpha_out), ("beta_out", beta_out), ("nvalid_out", nvalid_out)):
        if t is not None and t.numel() < tiles.numel():
            raise ValueError("%s is shorter than the tile list" % name)
    cap = 0 if out is None else out.numel() // 32
    if out is not None and out.dtype != torch.uint8:
        raise TypeError("out must be a uint8 tensor (32 bytes per record)")
    p = _SubParams(_MATCH[match], int(n_min), float(sci_wmin), float(ref_wmin), float(read_noise), float(gain), float(k_sigma), 0.0)
    n = C.c_size_t(0)
    f32 = torch.float32
    rc = load_library().argus_subtract_tiles(
        ctx._h, C.byref(lay), int(nside), _dev(sci_sum, f32, "sci_sum"), _dev(sci_wsum, f32, "sci_wsum"),
        _dev(ref_sum, f32, "ref_sum"), _dev(ref_wsum, f32, "ref_wsum"), C.byref(p), _dev(diff_out, f32, "diff_out"),
        _dev(sig_out, f32, "sig_out", allow_none=True), _dev(alpha_out, f32, "alpha_out", allow_none=True),
        _dev(beta_out, f32, "beta_out", allow_none=True), _dev(nvalid_out, torch.int32, "nvalid_out", allow_none=True),
        _dev(out, torch.uint8, "out", allow_none=True), cap, _dev(n_dev, torch.int64, "n_dev", allow_none=True),
        C.byref(n) if sync else None, _stream(stream))
    if rc == -6 and sync:
        raise ArgusError(rc, "argus_subtract_tiles", "n_candidates=%d" % n.value)
    _check(ctx, rc, "argus_subtract_tiles")
    return int(n.value) if sync else None


def argus_plan_info(ctx, stream=None) -> dict:
    s = _PlanStats()
    rc = load_library().argus_plan_info(ctx._h, C.byref(s), _stream(stream))
    _check(ctx, rc, "argus_plan_info")
    return {n: int(getattr(s, n)) for n, _ in _PlanStats._fields_}
