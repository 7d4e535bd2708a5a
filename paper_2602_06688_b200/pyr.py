"""Thin ctypes binding of libpyr (include/pyr.h): argument marshalling only.

Every step of the path (field build, FFT passes, mask, |.|^2 accumulation, rebin, slopes)
runs in the CUDA kernels of ``csrc/``; PyTorch supplies device memory and streams.  There is
no CPU fallback: if ``libpyr.so`` is missing or cannot be loaded, importing this module raises.

Names follow the C ABI (BASELINE.json:north_star): ``pyr_plan_create`` / ``pyr_compute`` /
``pyr_plan_destroy`` plus the extras of include/pyr.h; :class:`Plan` is a small RAII wrapper.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpyr.so")

PYR_OK, PYR_EINVAL, PYR_EUNSUPPORTED, PYR_ENOMEM, PYR_ECUDA = 0, 1, 2, 3, 4

EXPORTS = [
    "pyr_plan_create", "pyr_plan_create_points", "pyr_compute", "pyr_compute_host", "pyr_plan_destroy",
    "pyr_slopes_from_pixels", "pyr_slopes_from_pixels_static", "pyr_static_scratch_init", "pyr_plan_create_poly", "pyr_plan_set_double_roof",
    "pyr_compute_host_async", "pyr_host_wait", "pyr_plan_set_schedule",
    "pyr_plan_set_valid", "pyr_plan_set_mask_separable", "pyr_plan_set_mask", "pyr_plan_get_dims",
    "pyr_test_line_conv", "pyr_plan_launches_per_compute", "pyr_plan_set_profiling",
    "pyr_plan_last_kernel_ms", "pyr_kernel_name", "pyr_measure_fp32_peak", "pyr_last_error", "pyr_last_error_string",
]


class PyrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("libpyr error %d: %s" % (code, msg))
        self.code = code


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libpyr.so not found at %s -- build it with `python -m paper_2602_06688_b200.build` "
            "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
    ip = ctypes.POINTER(ctypes.c_int)
    L.pyr_plan_create.argtypes = [ci, ci, ci, cf, ci, ci]
    L.pyr_plan_create.restype = vp
    L.pyr_plan_create_points.argtypes = [ci, ci, ci, vp, vp, vp, ci, ci]
    L.pyr_plan_create_points.restype = vp
    L.pyr_compute.argtypes = [vp, vp, vp, vp, vp, vp]
    L.pyr_compute.restype = ci
    L.pyr_compute_host.argtypes = [vp, vp, vp, vp, vp, vp]
    L.pyr_compute_host.restype = ci
    L.pyr_compute_host_async.argtypes = [vp, vp, vp, vp, vp, ci]
    L.pyr_compute_host_async.restype = ci
    L.pyr_host_wait.argtypes = [vp, ci]
    L.pyr_host_wait.restype = ci
    L.pyr_plan_destroy.argtypes = [vp]
    L.pyr_plan_destroy.restype = None
    L.pyr_plan_create_poly.argtypes = [ci, ci, ci, cf, ci, vp, vp, ci, ci]
    L.pyr_plan_create_poly.restype = vp
    L.pyr_plan_set_schedule.argtypes = [vp, ci, ci]
    L.pyr_plan_set_schedule.restype = ci
    L.pyr_plan_set_double_roof.argtypes = [vp, ci, cf]
    L.pyr_plan_set_double_roof.restype = ci
    L.pyr_slopes_from_pixels.argtypes = [vp, vp, vp, vp]
    L.pyr_slopes_from_pixels.restype = ci
    L.pyr_slopes_from_pixels_static.argtypes = [ci, ci, vp, vp, ci, vp, vp]
    L.pyr_slopes_from_pixels_static.restype = ci
    L.pyr_static_scratch_init.argtypes = []
    L.pyr_static_scratch_init.restype = ci
    L.pyr_plan_set_valid.argtypes = [vp, vp]
    L.pyr_plan_set_valid.restype = ci
    L.pyr_plan_set_mask_separable.argtypes = [vp, vp, vp]
    L.pyr_plan_set_mask_separable.restype = ci
    L.pyr_plan_set_mask.argtypes = [vp, vp]
    L.pyr_plan_set_mask.restype = ci
    L.pyr_plan_get_dims.argtypes = [vp, ip, ip, ip]
    L.pyr_plan_get_dims.restype = ci
    L.pyr_test_line_conv.argtypes = [vp, vp, vp, ci, vp]
    L.pyr_test_line_conv.restype = ci
    L.pyr_plan_launches_per_compute.argtypes = [vp]
    L.pyr_plan_launches_per_compute.restype = ci
    L.pyr_plan_set_profiling.argtypes = [vp, ci]
    L.pyr_plan_set_profiling.restype = ci
    L.pyr_plan_last_kernel_ms.argtypes = [vp, ctypes.POINTER(cf), ci]
    L.pyr_plan_last_kernel_ms.restype = ci
    L.pyr_measure_fp32_peak.argtypes = [ctypes.POINTER(cf), ctypes.POINTER(cf)]
    L.pyr_measure_fp32_peak.restype = ci
    L.pyr_kernel_name.argtypes = [ci]
    L.pyr_kernel_name.restype = ctypes.c_char_p
    L.pyr_last_error.argtypes = []
    L.pyr_last_error.restype = ci
    L.pyr_last_error_string.argtypes = []
    L.pyr_last_error_string.restype = ctypes.c_char_p
    return L


lib = _load()


def last_error() -> tuple[int, str]:
    return lib.pyr_last_error(), (lib.pyr_last_error_string() or b"").decode()


def _check(rc: int) -> None:
    if rc != PYR_OK:
        raise PyrError(rc, last_error()[1])


def _dev_f32(t: torch.Tensor, shape, name: str) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("%s must be a contiguous float32 CUDA tensor" % name)
    if tuple(t.shape) != tuple(shape):
        raise ValueError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
    return t.data_ptr()


def _host_f32(t: torch.Tensor, shape, name: str) -> int:
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError("%s must be a contiguous float32 host tensor" % name)
    if tuple(t.shape) != tuple(shape):
        raise ValueError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
    return t.data_ptr()


def _stream_handle(stream) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


class Plan:
    """Owner of one ``pyr_plan`` (see ``pyr_plan_create`` in include/pyr.h)."""

    def __init__(self, N_pup: int, N_fft: int, n_mod: int, r_mod_lambda_over_D: float,
                 binning: int, batch: int, points=None, poly=None):
        """``points``: None for the modulation circle, else ``(ax, ay, weight_or_None)`` arrays of
        ``n_mod`` tilts in lambda/D (``pyr_plan_create_points``; ``r_mod_lambda_over_D`` is ignored).
        ``poly``: ``(ratio, weight_or_None)`` arrays over wavelengths (``pyr_plan_create_poly``)."""
        self._h = None
        if poly is not None:
            ratio = np.ascontiguousarray(poly[0], dtype=np.float32)
            wl = None if len(poly) < 2 or poly[1] is None else np.ascontiguousarray(poly[1], dtype=np.float32)
            if ratio.ndim != 1 or (wl is not None and wl.shape != ratio.shape):
                raise ValueError("poly arrays must be 1-D and of equal length")
            h = lib.pyr_plan_create_poly(int(N_pup), int(N_fft), int(n_mod), float(r_mod_lambda_over_D), int(ratio.shape[0]),
                                         ratio.ctypes.data, None if wl is None else wl.ctypes.data, int(binning), int(batch))
        elif points is None:
            h = lib.pyr_plan_create(int(N_pup), int(N_fft), int(n_mod), float(r_mod_lambda_over_D),
                                    int(binning), int(batch))
        else:
            ax = np.ascontiguousarray(points[0], dtype=np.float32)
            ay = np.ascontiguousarray(points[1], dtype=np.float32)
            w = None if len(points) < 3 or points[2] is None else np.ascontiguousarray(points[2], dtype=np.float32)
            if ax.shape != (int(n_mod),) or ay.shape != (int(n_mod),) or (w is not None and w.shape != (int(n_mod),)):
                raise ValueError("points arrays must have n_mod entries")
            h = lib.pyr_plan_create_points(int(N_pup), int(N_fft), int(n_mod), ax.ctypes.data, ay.ctypes.data,
                                           None if w is None else w.ctypes.data, int(binning), int(batch))
        if not h:
            raise PyrError(*last_error())
        self._h = h
        self.N_pup, self.N_fft, self.n_mod = int(N_pup), int(N_fft), int(n_mod)
        self.r_mod, self.binning, self.batch = float(r_mod_lambda_over_D), int(binning), int(batch)
        nd, nq, nv = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        _check(lib.pyr_plan_get_dims(h, ctypes.byref(nd), ctypes.byref(nq), ctypes.byref(nv)))
        self.N_det, self.N_q = nd.value, nq.value

    @classmethod
    def from_points(cls, N_pup, N_fft, ax, ay, weight, binning, batch):
        return cls(N_pup, N_fft, len(ax), 0.0, binning, batch, points=(ax, ay, weight))

    # -- lifetime
    def destroy(self) -> None:
        if self._h:
            lib.pyr_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    # -- queries
    @property
    def n_valid(self) -> int:
        nv = ctypes.c_int()
        _check(lib.pyr_plan_get_dims(self._h, None, None, ctypes.byref(nv)))
        return nv.value

    @property
    def launches_per_compute(self) -> int:
        return lib.pyr_plan_launches_per_compute(self._h)

    # -- measurement hooks
    def set_profiling(self, enable: bool) -> None:
        _check(lib.pyr_plan_set_profiling(self._h, 1 if enable else 0))

    def last_kernel_ms(self) -> dict:
        """Device time (ms) of every kernel of the last profiled ``compute`` (waits for it)."""
        buf = (ctypes.c_float * 8)()
        n = lib.pyr_plan_last_kernel_ms(self._h, buf, 8)
        if n < 0:
            raise PyrError(*last_error())
        return {lib.pyr_kernel_name(i).decode(): float(buf[i]) for i in range(n)}

    # -- tables
    def set_valid(self, valid) -> None:
        v = np.ascontiguousarray(valid, dtype=np.uint8)
        if v.shape != (self.N_q, self.N_q):
            raise ValueError("valid has shape %s, expected %s" % (v.shape, (self.N_q, self.N_q)))
        _check(lib.pyr_plan_set_valid(self._h, v.ctypes.data))

    def set_schedule(self, l2_resident: bool, j_per_chunk: int = 0) -> None:
        """``pyr_plan_set_schedule``: per-chunk passes with R as an L2-resident ring (N_fft = 2048)."""
        _check(lib.pyr_plan_set_schedule(self._h, int(bool(l2_resident)), int(j_per_chunk)))

    def set_double_roof(self, kappa, enable=True) -> None:
        """``pyr_plan_set_double_roof``: ModulatedDoubleRoof with the inter-plane factor exp(i pi kappa rho^2)."""
        _check(lib.pyr_plan_set_double_roof(self._h, int(bool(enable)), float(kappa)))

    def set_mask_separable(self, gx=None, gy=None) -> None:
        if gx is None and gy is None:
            _check(lib.pyr_plan_set_mask_separable(self._h, None, None))
            return
        a = np.ascontiguousarray(np.asarray(gx, dtype=np.complex64)).view(np.float32)
        b = np.ascontiguousarray(np.asarray(gy, dtype=np.complex64)).view(np.float32)
        if a.shape != (2 * self.N_fft,) or b.shape != (2 * self.N_fft,):
            raise ValueError("gx, gy must have N_fft complex entries")
        _check(lib.pyr_plan_set_mask_separable(self._h, a.ctypes.data, b.ctypes.data))

    def set_mask(self, mask=None) -> None:
        """General complex [N_fft][N_fft] mask (natural DFT order, mask[v][u]); None restores the previous one."""
        if mask is None:
            _check(lib.pyr_plan_set_mask(self._h, None))
            return
        m = np.ascontiguousarray(np.asarray(mask, dtype=np.complex64))
        if m.shape != (self.N_fft, self.N_fft):
            raise ValueError("mask must be [N_fft][N_fft] complex")
        _check(lib.pyr_plan_set_mask(self._h, m.view(np.float32).ctypes.data))

    # -- the hot call
    def empty_outputs(self, device="cuda"):
        I = torch.empty((self.batch, self.N_det, self.N_det), dtype=torch.float32, device=device)
        s = torch.empty((self.batch, 2, self.N_q, self.N_q), dtype=torch.float32, device=device)
        return I, s

    def compute(self, amp, phase, out_intensity=None, out_slopes=None, stream=None) -> None:
        """``pyr_compute``: device tensors, asynchronous on ``stream`` (default: current)."""
        shp = (self.batch, self.N_pup, self.N_pup)
        a = _dev_f32(amp, shp, "amp")
        p = _dev_f32(phase, shp, "phase")
        oi = None if out_intensity is None else _dev_f32(
            out_intensity, (self.batch, self.N_det, self.N_det), "out_intensity")
        os_ = None if out_slopes is None else _dev_f32(
            out_slopes, (self.batch, 2, self.N_q, self.N_q), "out_slopes")
        _check(lib.pyr_compute(self._h, a, p, oi, os_, _stream_handle(stream)))

    def slopes_from_pixels(self, pixels, out_slopes, stream=None) -> None:
        """``pyr_slopes_from_pixels``: PyrSlopec on a detector frame [B][N_det][N_det] (device tensors)."""
        px = _dev_f32(pixels, (self.batch, self.N_det, self.N_det), "pixels")
        os_ = _dev_f32(out_slopes, (self.batch, 2, self.N_q, self.N_q), "out_slopes")
        _check(lib.pyr_slopes_from_pixels(self._h, px, os_, _stream_handle(stream)))

    def compute_host(self, amp, phase, out_intensity=None, out_slopes=None, stream=None) -> None:
        """``pyr_compute_host``: host tensors in and out; returns when the results are there."""
        shp = (self.batch, self.N_pup, self.N_pup)
        a = _host_f32(amp, shp, "amp")
        p = _host_f32(phase, shp, "phase")
        oi = None if out_intensity is None else _host_f32(
            out_intensity, (self.batch, self.N_det, self.N_det), "out_intensity")
        os_ = None if out_slopes is None else _host_f32(
            out_slopes, (self.batch, 2, self.N_q, self.N_q), "out_slopes")
        _check(lib.pyr_compute_host(self._h, a, p, oi, os_, _stream_handle(stream)))

    def compute_host_async(self, amp, phase, out_intensity=None, out_slopes=None, slot=0) -> None:
        """``pyr_compute_host_async``: enqueue H2D, kernels and D2H of one call on staging slot 0 or 1 (pinned host
        tensors); the results are there after ``host_wait(slot)``."""
        shp = (self.batch, self.N_pup, self.N_pup)
        a = _host_f32(amp, shp, "amp")
        p = _host_f32(phase, shp, "phase")
        oi = None if out_intensity is None else _host_f32(
            out_intensity, (self.batch, self.N_det, self.N_det), "out_intensity")
        os_ = None if out_slopes is None else _host_f32(
            out_slopes, (self.batch, 2, self.N_q, self.N_q), "out_slopes")
        _check(lib.pyr_compute_host_async(self._h, a, p, oi, os_, int(slot)))

    def host_wait(self, slot=0) -> None:
        _check(lib.pyr_host_wait(self._h, int(slot)))

    def test_line_conv(self, lines: torch.Tensor, stream=None) -> torch.Tensor:
        """Test-only: ``IDFT(g_x . DFT(zero-pad(line)))/N`` per line.  lines: complex64
        CUDA tensor [nlines][N_pup]; returns complex64 [nlines][N_fft]."""
        if not (lines.is_cuda and lines.dtype == torch.complex64 and lines.is_contiguous()
                and lines.dim() == 2 and lines.shape[1] == self.N_pup):
            raise TypeError("lines must be a contiguous complex64 CUDA tensor [nlines][N_pup]")
        out = torch.empty((lines.shape[0], self.N_fft), dtype=torch.complex64, device=lines.device)
        _check(lib.pyr_test_line_conv(self._h, lines.data_ptr(), out.data_ptr(), int(lines.shape[0]),
                                      _stream_handle(stream)))
        return out


def static_scratch_init() -> None:
    """``pyr_static_scratch_init``: resolve the static scratch array's address on the current device."""
    _check(lib.pyr_static_scratch_init())


def slopes_from_pixels_static(pixels, valid, n_valid, out_slopes, stream=None) -> None:
    """``pyr_slopes_from_pixels_static``: slopes of detector frames without a plan and without any allocation
    (argument marshalling only).  pixels [B][N_det][N_det] float32, valid [N_q][N_q] uint8, out_slopes
    [B][2][N_q][N_q] float32, all CUDA tensors; n_valid = the number of non-zero entries of valid."""
    if not (isinstance(pixels, torch.Tensor) and pixels.dim() == 3 and pixels.shape[1] == pixels.shape[2]):
        raise ValueError("pixels must be [B][N_det][N_det]")
    B, Nd = int(pixels.shape[0]), int(pixels.shape[1])
    px = _dev_f32(pixels, (B, Nd, Nd), "pixels")
    if not (isinstance(valid, torch.Tensor) and valid.is_cuda and valid.dtype == torch.uint8 and valid.is_contiguous()
            and tuple(valid.shape) == (Nd // 2, Nd // 2)):
        raise TypeError("valid must be a contiguous uint8 CUDA tensor of shape [N_q][N_q]")
    os_ = _dev_f32(out_slopes, (B, 2, Nd // 2, Nd // 2), "out_slopes")
    _check(lib.pyr_slopes_from_pixels_static(Nd, B, px, valid.data_ptr(), int(n_valid), os_, _stream_handle(stream)))


def measure_fp32_peak():
    """``pyr_measure_fp32_peak``: (TFLOP/s, effective SM MHz) of the packed-FMA microbenchmark."""
    tf, mhz = ctypes.c_float(), ctypes.c_float()
    _check(lib.pyr_measure_fp32_peak(ctypes.byref(tf), ctypes.byref(mhz)))
    return float(tf.value), float(mhz.value)


# C-ABI names, for callers who want the flat interface.
def pyr_plan_create(N_pup, N_fft, n_mod, r_mod_lambda_over_D, binning, batch) -> Plan:
    return Plan(N_pup, N_fft, n_mod, r_mod_lambda_over_D, binning, batch)


def pyr_compute(plan: Plan, amp, phase, out_intensity, out_slopes, stream=None) -> None:
    plan.compute(amp, phase, out_intensity, out_slopes, stream)


def pyr_plan_destroy(plan: Plan) -> None:
    plan.destroy()
