"""ctypes loader for the Shack-Hartmann CPU oracle (``oracle/sh_oracle.c``).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/`` and ``bench.py``'s extras may import it.  All
arithmetic lives in the C file; this module builds it with gcc, loads it and marshals NumPy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sh_oracle.c")
_LIB = os.path.join(_HERE, "libshoracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c99", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        fp = ctypes.POINTER(ctypes.c_float)
        L.sho_spot.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp]
        L.sho_spot.restype = None
        L.sh_oracle_compute.argtypes = [ctypes.c_int] * 5 + [fp, fp, dp, dp, dp]
        L.sh_oracle_compute.restype = ctypes.c_int
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def spot(e: np.ndarray, F: int) -> np.ndarray:
    """S = |DFT2_F(zero-pad(e))|^2 / F^2 of one complex p x p patch."""
    e = np.ascontiguousarray(e, dtype=np.complex128)
    p = e.shape[0]
    assert e.shape == (p, p)
    S = np.empty((F, F), dtype=np.float64)
    lib().sho_spot(p, int(F), _dptr(e.view(np.float64)), _dptr(S))
    return S


def compute(P, n_sub, F, bs, amp, phase, want_spots=False):
    """Returns (slopes [B][2][n_sub][n_sub], flux [B][n_sub][n_sub], spots or None)."""
    amp = np.ascontiguousarray(amp, dtype=np.float32)
    phase = np.ascontiguousarray(phase, dtype=np.float32)
    if amp.ndim == 2:
        amp, phase = amp[None], phase[None]
    B = amp.shape[0]
    assert amp.shape == (B, P, P) and phase.shape == (B, P, P)
    npix = F // bs
    s = np.empty((B, 2, n_sub, n_sub), dtype=np.float64)
    fl = np.empty((B, n_sub, n_sub), dtype=np.float64)
    sp = np.empty((B, n_sub, n_sub, npix, npix), dtype=np.float64) if want_spots else None
    fpt = ctypes.POINTER(ctypes.c_float)
    rc = lib().sh_oracle_compute(int(P), int(n_sub), int(F), int(bs), int(B), amp.ctypes.data_as(fpt),
                                 phase.ctypes.data_as(fpt), _dptr(s), _dptr(fl), _dptr(sp) if sp is not None else None)
    if rc:
        raise ValueError("sh_oracle_compute failed rc=%d" % rc)
    return s, fl, sp
