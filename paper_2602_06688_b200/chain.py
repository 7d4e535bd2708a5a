"""ctypes binding of the steps either side of the sensor (include/chain.h, part of libpyr.so): argument
marshalling only.  PyTorch supplies device memory and streams.  Raises at import if the library is missing:
there is no CPU fallback."""
from __future__ import annotations

import ctypes

import numpy as np
import torch

from . import pyr as _pyr

EXPORTS = [
    "atmo_plan_create", "atmo_plan_set_weights", "atmo_propagate", "atmo_plan_destroy",
    "ccd_plan_create", "ccd_integrate", "ccd_reset", "ccd_plan_destroy", "ccd_test_philox",
    "pupdata_from_frame",
    "modalrec_plan_create", "modalrec_compute", "modalrec_plan_destroy",
    "chain_last_error", "chain_last_error_string",
]

lib = _pyr.lib
_vp, _ci, _cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
_ll, _ull, _cu = ctypes.c_longlong, ctypes.c_ulonglong, ctypes.c_uint
lib.atmo_plan_create.argtypes = [_ci] * 4
lib.atmo_plan_create.restype = _vp
lib.atmo_plan_set_weights.argtypes = [_vp, _vp]
lib.atmo_plan_set_weights.restype = _ci
lib.atmo_propagate.argtypes = [_vp, _vp, _vp, _vp, _vp]
lib.atmo_propagate.restype = _ci
lib.atmo_plan_destroy.argtypes = [_vp]
lib.atmo_plan_destroy.restype = None
lib.ccd_plan_create.argtypes = [_ll, _ci, _ci, _ci, _cf, _cf, _ci, _ull]
lib.ccd_plan_create.restype = _vp
lib.ccd_integrate.argtypes = [_vp, _vp, _cf, _vp, ctypes.POINTER(_ci), _vp]
lib.ccd_integrate.restype = _ci
lib.ccd_reset.argtypes = [_vp, _vp]
lib.ccd_reset.restype = _ci
lib.ccd_plan_destroy.argtypes = [_vp]
lib.ccd_plan_destroy.restype = None
lib.ccd_test_philox.argtypes = [_ull, _cu, _ll, _vp, _vp]
lib.ccd_test_philox.restype = _ci
lib.pupdata_from_frame.argtypes = [_ci, _vp, _cf, _vp, _vp]
lib.pupdata_from_frame.restype = _ci
lib.modalrec_plan_create.argtypes = [_ci, _ci, _vp, _vp, _ci]
lib.modalrec_plan_create.restype = _vp
lib.modalrec_compute.argtypes = [_vp, _vp, _vp, _vp]
lib.modalrec_compute.restype = _ci
lib.modalrec_plan_destroy.argtypes = [_vp]
lib.modalrec_plan_destroy.restype = None
lib.chain_last_error.argtypes = []
lib.chain_last_error.restype = _ci
lib.chain_last_error_string.argtypes = []
lib.chain_last_error_string.restype = ctypes.c_char_p


class ChainError(RuntimeError):
    pass


def _fail():
    raise ChainError("libpyr (chain) error %d: %s" % (lib.chain_last_error(), lib.chain_last_error_string().decode()))


def _check(rc):
    if rc:
        _fail()


def _dev(t, shape, name, dtype=torch.float32):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()
            and tuple(t.shape) == tuple(shape)):
        raise ValueError("%s must be a contiguous %s CUDA tensor of shape %s" % (name, dtype, tuple(shape)))
    return t.data_ptr()


def _st(stream):
    return (stream if stream is not None else torch.cuda.current_stream()).cuda_stream


class _Owner:
    _destroy = None

    def destroy(self):
        if getattr(self, "_h", None):
            type(self)._destroy(self._h)
            self._h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Atmo(_Owner):
    """``atmo_plan``: shifted periodic phase screens -> pupil phase (AtmoEvolution + AtmoPropagation)."""
    _destroy = lib.atmo_plan_destroy

    def __init__(self, n_layers, screen_side, N_pup, batch, weights=None):
        self._h = lib.atmo_plan_create(int(n_layers), int(screen_side), int(N_pup), int(batch))
        if not self._h:
            _fail()
        self.L, self.S, self.P, self.B = int(n_layers), int(screen_side), int(N_pup), int(batch)
        if weights is not None:
            w = np.ascontiguousarray(weights, dtype=np.float32)
            assert w.shape == (self.L,)
            _check(lib.atmo_plan_set_weights(self._h, w.ctypes.data))

    def propagate(self, screens, shift_yx, out_phase, stream=None):
        sh = np.ascontiguousarray(shift_yx, dtype=np.float64)
        if sh.shape != (self.B, self.L, 2):
            raise ValueError("shift_yx must be [B][L][2]")
        _check(lib.atmo_propagate(self._h, _dev(screens, (self.L, self.S, self.S), "screens"), sh.ctypes.data,
                                  _dev(out_phase, (self.B, self.P, self.P), "out_phase"), _st(stream)))


class CCD(_Owner):
    """``ccd_plan``: integration, photon and readout noise, ADC."""
    _destroy = lib.ccd_plan_destroy

    def __init__(self, shape, n_int=1, photon_noise=True, readout_noise=True, readout_level=0.4, adu_gain=0.0,
                 n_bits=16, seed=1):
        self.shape = tuple(int(v) for v in shape)
        n = int(np.prod(self.shape))
        self._h = lib.ccd_plan_create(n, int(n_int), int(bool(photon_noise)), int(bool(readout_noise)),
                                      float(readout_level), float(adu_gain), int(n_bits), int(seed))
        if not self._h:
            _fail()

    def integrate(self, intensity, flux_gain, out_pixels, stream=None) -> bool:
        """One step; True when ``out_pixels`` was written (a frame was read out)."""
        ready = _ci(0)
        _check(lib.ccd_integrate(self._h, _dev(intensity, self.shape, "intensity"), float(flux_gain),
                                 None if out_pixels is None else _dev(out_pixels, self.shape, "out_pixels"),
                                 ctypes.byref(ready), _st(stream)))
        return bool(ready.value)

    def reset(self, stream=None):
        _check(lib.ccd_reset(self._h, _st(stream)))


def philox_words(seed, frame, n, stream=None):
    """Test-only: the generator's raw output for counters (i, frame, 0, 0), i < n: uint32 [n][4] (as int32 tensor bits)."""
    out = torch.empty((int(n), 4), dtype=torch.int32, device="cuda")
    _check(lib.ccd_test_philox(int(seed), int(frame), int(n), out.data_ptr(), _st(stream)))
    return out


def pupdata_from_frame(ref_frame, threshold, stream=None):
    """``pupdata_from_frame``: uint8 [N_q][N_q] validity map (host) from a device reference frame [N_det][N_det]."""
    Nd = int(ref_frame.shape[0])
    valid = np.empty((Nd // 2, Nd // 2), dtype=np.uint8)
    _check(lib.pupdata_from_frame(Nd, _dev(ref_frame, (Nd, Nd), "ref_frame"), float(threshold), valid.ctypes.data, _st(stream)))
    return valid


class Modalrec(_Owner):
    """``modalrec_plan``: modes = R . (valid slopes)."""
    _destroy = lib.modalrec_plan_destroy

    def __init__(self, recmat, valid, batch):
        v = np.ascontiguousarray(valid, dtype=np.uint8)
        R = np.ascontiguousarray(recmat, dtype=np.float32)
        self.N_q, self.n_modes, self.B = int(v.shape[0]), int(R.shape[0]), int(batch)
        if v.shape != (self.N_q, self.N_q) or R.shape != (self.n_modes, 2 * int(v.sum())):
            raise ValueError("recmat must be [n_modes][2 n_valid]")
        self._h = lib.modalrec_plan_create(self.n_modes, self.N_q, v.ctypes.data, R.ctypes.data, self.B)
        if not self._h:
            _fail()

    def compute(self, slopes, out_modes, stream=None):
        _check(lib.modalrec_compute(self._h, _dev(slopes, (self.B, 2, self.N_q, self.N_q), "slopes"),
                                    _dev(out_modes, (self.B, self.n_modes), "out_modes"), _st(stream)))
