"""ctypes loader for ``oracle/chain_oracle.c`` (atmosphere propagation, CCD, PupData, Modalrec: SURVEY.md 8(f) f3).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/`` and ``bench.py``'s cpu legs may import this module; it
imports nothing from ``paper_2602_06688_b200``.  All arithmetic lives in the C file; this module builds it
with gcc (``-ffp-contract=off``: the float32 noise model must not be re-associated or fused), loads it and
marshals NumPy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "chain_oracle.c")
_LIB = os.path.join(_HERE, "libchainoracle.so")
_lib = None

_f, _d, _i, _u32, _u64 = ctypes.c_float, ctypes.c_double, ctypes.c_int, ctypes.c_uint32, ctypes.c_uint64
_fp, _dp, _bp, _up = (ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double),
                      ctypes.POINTER(ctypes.c_ubyte), ctypes.POINTER(ctypes.c_uint32))


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.chain_oracle_atmo.argtypes = [_i, _i, _i, _i, _fp, _dp, _dp, _dp]
        L.chain_oracle_atmo.restype = _i
        L.cho_philox4x32_10.argtypes = [_up, _up, _up]
        L.cho_philox4x32_10.restype = None
        for name, args in (("cho_u01", [_u32]), ("cho_exp_neg", [_f]), ("cho_log", [_f]), ("cho_cos2pi", [_f]),
                           ("cho_normal", [_f, _f]), ("cho_poisson", [_f, _f, _f])):
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = _f
        L.chain_oracle_ccd.argtypes = [ctypes.c_longlong, _fp, _fp, _f, _i, _i, _i, _f, _f, _i, _u64, _u32, _fp]
        L.chain_oracle_ccd.restype = _i
        L.chain_oracle_pupdata.argtypes = [_i, _fp, _f, _bp]
        L.chain_oracle_pupdata.restype = _i
        L.chain_oracle_modalrec.argtypes = [_i, _i, _i, _bp, _fp, _fp, _dp]
        L.chain_oracle_modalrec.restype = _i
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def atmo(screens, shift_yx, P, weights=None):
    """phase [B][P][P] (float64) from screens [L][S][S] (float32) displaced by shift_yx [B][L][2] pixels."""
    screens = np.ascontiguousarray(screens, dtype=np.float32)
    shift_yx = np.ascontiguousarray(shift_yx, dtype=np.float64)
    L, S, _ = screens.shape
    B = shift_yx.shape[0]
    assert screens.shape == (L, S, S) and shift_yx.shape == (B, L, 2)
    w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float64)
    out = np.empty((B, P, P), dtype=np.float64)
    rc = lib().chain_oracle_atmo(L, S, int(P), B, _p(screens, _fp), _p(w, _dp) if w is not None else None,
                                 _p(shift_yx, _dp), _p(out, _dp))
    if rc:
        raise ValueError("chain_oracle_atmo failed rc=%d" % rc)
    return out


def philox(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    o = np.empty(4, dtype=np.uint32)
    lib().cho_philox4x32_10(_p(c, _up), _p(k, _up), _p(o, _up))
    return o


def u01(x):
    return float(lib().cho_u01(int(x)))


def exp_neg(x):
    return float(lib().cho_exp_neg(float(x)))


def log(x):
    return float(lib().cho_log(float(x)))


def cos2pi(x):
    return float(lib().cho_cos2pi(float(x)))


def normal(ua, ub):
    return float(lib().cho_normal(float(ua), float(ub)))


def poisson(lam, ua, ub):
    return float(lib().cho_poisson(float(lam), float(ua), float(ub)))


class CCD:
    """State of one detector: the float32 accumulator and the frame counter (chain_oracle_ccd)."""

    def __init__(self, shape, n_int=1, photon_noise=True, readout_noise=True, readout_level=0.4, adu_gain=0.0,
                 n_bits=16, seed=1):
        self.acc = np.zeros(shape, dtype=np.float32)
        self.n_int, self.step, self.frame = int(n_int), 0, 0
        self.cfg = (int(bool(photon_noise)), int(bool(readout_noise)), float(readout_level), float(adu_gain), int(n_bits), int(seed))

    def integrate(self, D, gain):
        """One step; returns the float32 frame when the integration completes, else None."""
        D = np.ascontiguousarray(D, dtype=np.float32)
        assert D.shape == self.acc.shape
        self.step += 1
        ready = self.step % self.n_int == 0
        out = np.empty_like(self.acc) if ready else None
        pn, rn, sig, adu, nb, seed = self.cfg
        rc = lib().chain_oracle_ccd(self.acc.size, _p(self.acc, _fp), _p(D, _fp), float(gain), int(ready), pn, rn, sig,
                                    adu, nb, seed, self.frame, _p(out, _fp) if ready else None)
        if rc:
            raise ValueError("chain_oracle_ccd failed rc=%d" % rc)
        if ready:
            self.frame += 1
        return out


def pupdata(ref, thr):
    ref = np.ascontiguousarray(ref, dtype=np.float32)
    Nd = ref.shape[0]
    valid = np.empty((Nd // 2, Nd // 2), dtype=np.uint8)
    rc = lib().chain_oracle_pupdata(Nd, _p(ref, _fp), float(thr), _p(valid, _bp))
    if rc:
        raise ValueError("chain_oracle_pupdata failed rc=%d" % rc)
    return valid


def modalrec(R, valid, slopes):
    """modes [B][n_modes] (float64) from dense slopes [B][2][Nq][Nq] (float32)."""
    valid = np.ascontiguousarray(valid, dtype=np.uint8)
    Nq = valid.shape[0]
    slopes = np.ascontiguousarray(slopes, dtype=np.float32)
    B = slopes.shape[0]
    R = np.ascontiguousarray(R, dtype=np.float32)
    n_modes = R.shape[0]
    assert slopes.shape == (B, 2, Nq, Nq) and R.shape == (n_modes, 2 * int(valid.sum()))
    out = np.empty((B, n_modes), dtype=np.float64)
    rc = lib().chain_oracle_modalrec(n_modes, Nq, B, _p(valid, _bp), _p(R, _fp), _p(slopes, _fp), _p(out, _dp))
    if rc:
        raise ValueError("chain_oracle_modalrec failed rc=%d" % rc)
    return out
