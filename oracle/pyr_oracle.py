"""ctypes loader for the CPU oracle (``oracle/pyr_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this module.  It
imports nothing from ``paper_2602_06688_b200`` and the CUDA library imports nothing from
here.  All arithmetic lives in the C file; this module only builds it with gcc, loads it and
marshals NumPy arrays.

The operation is the one named by BASELINE.json:north_star (paper: ``ModulatedPyramid`` +
``PyrSlopec``; parameters PAPER.md:528-556) in the reading of
SURVEY.md section 8(c).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pyr_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile ``pyr_oracle.c`` to ``liboracle.so`` next to it (gcc, -O2)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-fPIC", "-shared", "-pthread", "-std=c99", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        fp = ctypes.POINTER(ctypes.c_float)
        bp = ctypes.POINTER(ctypes.c_ubyte)
        L.pyro_dft_direct.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
        L.pyro_dft_direct.restype = None
        L.pyro_fft1d.argtypes = [ctypes.c_int, ctypes.c_int, dp]
        L.pyro_fft1d.restype = ctypes.c_int
        L.pyro_fft2d.argtypes = [ctypes.c_int, ctypes.c_int, dp]
        L.pyro_fft2d.restype = ctypes.c_int
        L.pyro_pyramid_mask.argtypes = [ctypes.c_int, dp]
        L.pyro_pyramid_mask.restype = None
        L.pyro_default_valid.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, bp]
        L.pyro_default_valid.restype = None
        L.pyro_rebin.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
        L.pyro_rebin.restype = None
        L.pyro_slopes.argtypes = [ctypes.c_int, dp, bp, dp]
        L.pyro_slopes.restype = None
        L.pyr_oracle_compute.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            fp, fp, dp, bp, dp, dp, dp, ctypes.c_int,
        ]
        L.pyr_oracle_compute.restype = ctypes.c_int
        L.pyr_oracle_compute_points.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, ctypes.c_int, ctypes.c_int,
            fp, fp, dp, bp, dp, dp, dp, ctypes.c_int,
        ]
        L.pyr_oracle_compute_points.restype = ctypes.c_int
        L.pyr_oracle_compute_poly.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, dp, dp, ctypes.c_int, ctypes.c_int,
            fp, fp, dp, bp, dp, dp, dp, ctypes.c_int,
        ]
        L.pyr_oracle_compute_poly.restype = ctypes.c_int
        L.pyr_oracle_compute_double_roof.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            fp, fp, bp, dp, dp, dp, ctypes.c_int,
        ]
        L.pyr_oracle_compute_double_roof.restype = ctypes.c_int
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c2ri(z: np.ndarray) -> np.ndarray:
    z = np.ascontiguousarray(z, dtype=np.complex128)
    return z.view(np.float64).reshape(z.shape + (2,)).copy()


def _ri2c(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a).view(np.complex128).reshape(a.shape[:-1])


def dft_direct(x: np.ndarray, sign: int) -> np.ndarray:
    """O(n^2) direct DFT of a 1-D complex array, unscaled, exponent sign ``sign``."""
    a = _c2ri(np.asarray(x).ravel())
    out = np.empty_like(a)
    lib().pyro_dft_direct(a.shape[0], int(sign), _dptr(a), _dptr(out))
    return _ri2c(out)


def fft1d(x: np.ndarray, sign: int) -> np.ndarray:
    """The oracle's own 1-D transform (radix-2 FFT for powers of two), unscaled."""
    a = _c2ri(np.asarray(x).ravel())
    rc = lib().pyro_fft1d(a.shape[0], int(sign), _dptr(a))
    if rc:
        raise ValueError("pyro_fft1d failed rc=%d" % rc)
    return _ri2c(a)


def fft2d(x: np.ndarray, sign: int) -> np.ndarray:
    """The oracle's own 2-D transform of an n x n array (n a power of two), unscaled."""
    x = np.asarray(x)
    assert x.ndim == 2 and x.shape[0] == x.shape[1]
    a = _c2ri(x)
    rc = lib().pyro_fft2d(x.shape[0], int(sign), _dptr(a))
    if rc:
        raise ValueError("pyro_fft2d failed rc=%d" % rc)
    return _ri2c(a)


def pyramid_mask(n: int) -> np.ndarray:
    a = np.empty((n, n, 2), dtype=np.float64)
    lib().pyro_pyramid_mask(int(n), _dptr(a))
    return _ri2c(a)


def default_valid(P: int, N: int, b: int) -> np.ndarray:
    Nq = N // b // 2
    v = np.zeros((Nq, Nq), dtype=np.uint8)
    lib().pyro_default_valid(int(P), int(N), int(b), v.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)))
    return v


def rebin(I: np.ndarray, b: int) -> np.ndarray:
    I = np.ascontiguousarray(I, dtype=np.float64)
    N = I.shape[0]
    D = np.empty((N // b, N // b), dtype=np.float64)
    lib().pyro_rebin(N, int(b), _dptr(I), _dptr(D))
    return D


def slopes_from_D(D: np.ndarray, valid: np.ndarray) -> np.ndarray:
    D = np.ascontiguousarray(D, dtype=np.float64)
    Nd = D.shape[0]
    valid = np.ascontiguousarray(valid, dtype=np.uint8)
    s = np.empty((2, Nd // 2, Nd // 2), dtype=np.float64)
    lib().pyro_slopes(Nd, _dptr(D), valid.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)), _dptr(s))
    return s


def compute(P, N, M, r, b, amp, phase, mask=None, valid=None, want_full=False, nthreads=None, points=None,
            poly=None, double_roof=None):
    """Run the whole path.  ``amp``/``phase``: float32 [B][P][P].  ``points``: None for the modulation
    circle (M, r), else ``(ax, ay, w_or_None)`` arrays of M tilts in lambda/D and weights.  ``poly``:
    ``(ratio, weight_or_None)`` arrays over wavelengths (PolyCromPyramid, ratio = lambda_0 / lambda).
    ``double_roof``: kappa of the ModulatedDoubleRoof (two roof prisms in two focal planes).

    Returns ``(D, slopes, I_full_or_None)`` as float64 arrays of shapes
    ``[B][N/b][N/b]``, ``[B][2][Nq][Nq]``, ``[B][N][N]``.
    """
    amp = np.ascontiguousarray(amp, dtype=np.float32)
    phase = np.ascontiguousarray(phase, dtype=np.float32)
    if amp.ndim == 2:
        amp = amp[None]
        phase = phase[None]
    B = amp.shape[0]
    assert amp.shape == (B, P, P) and phase.shape == (B, P, P)
    Nd = N // b
    Nq = Nd // 2
    D = np.empty((B, Nd, Nd), dtype=np.float64)
    S = np.empty((B, 2, Nq, Nq), dtype=np.float64)
    If = np.empty((B, N, N), dtype=np.float64) if want_full else None
    mk = None
    if mask is not None:
        mk = _c2ri(np.asarray(mask))
        assert mk.shape == (N, N, 2)
    vm = None
    if valid is not None:
        vm = np.ascontiguousarray(valid, dtype=np.uint8)
        assert vm.shape == (Nq, Nq)
    if nthreads is None:
        nthreads = max(1, min(os.cpu_count() or 1, 64))
    fpt = ctypes.POINTER(ctypes.c_float)
    common = (
        amp.ctypes.data_as(fpt), phase.ctypes.data_as(fpt),
        _dptr(mk) if mk is not None else None,
        vm.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)) if vm is not None else None,
        _dptr(If) if If is not None else None, _dptr(D), _dptr(S), int(nthreads),
    )
    if double_roof is not None:
        assert mask is None and points is None and poly is None
        rc = lib().pyr_oracle_compute_double_roof(int(P), int(N), int(M), float(r), float(double_roof), int(b), int(B),
                                                  common[0], common[1], *common[3:])
    elif poly is not None:
        assert points is None
        ratio = np.ascontiguousarray(poly[0], dtype=np.float64)
        wl = None if len(poly) < 2 or poly[1] is None else np.ascontiguousarray(poly[1], dtype=np.float64)
        assert ratio.ndim == 1 and (wl is None or wl.shape == ratio.shape)
        rc = lib().pyr_oracle_compute_poly(int(P), int(N), int(M), float(r), int(ratio.shape[0]), _dptr(ratio),
                                           _dptr(wl) if wl is not None else None, int(b), int(B), *common)
    elif points is None:
        rc = lib().pyr_oracle_compute(int(P), int(N), int(M), float(r), int(b), int(B), *common)
    else:
        ax = np.ascontiguousarray(points[0], dtype=np.float64)
        ay = np.ascontiguousarray(points[1], dtype=np.float64)
        w = None if len(points) < 3 or points[2] is None else np.ascontiguousarray(points[2], dtype=np.float64)
        assert ax.shape == (M,) and ay.shape == (M,) and (w is None or w.shape == (M,))
        rc = lib().pyr_oracle_compute_points(int(P), int(N), int(M), _dptr(ax), _dptr(ay),
                                             _dptr(w) if w is not None else None, int(b), int(B), *common)
    if rc:
        raise ValueError("pyr_oracle_compute failed rc=%d" % rc)
    return D, S, If
