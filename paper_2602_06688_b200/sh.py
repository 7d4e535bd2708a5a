"""ctypes binding of the Shack-Hartmann path of libpyr.so (include/sh.h): argument marshalling only.
PyTorch supplies device memory and streams.  Raises at import if the library is missing: there is no
CPU fallback."""
from __future__ import annotations

import ctypes

import torch

from . import pyr as _pyr

EXPORTS = ["sh_plan_create", "sh_compute", "sh_plan_destroy", "sh_last_error", "sh_last_error_string"]

lib = _pyr.lib
_vp, _ci = ctypes.c_void_p, ctypes.c_int
lib.sh_plan_create.argtypes = [_ci] * 5
lib.sh_plan_create.restype = _vp
lib.sh_compute.argtypes = [_vp] * 7
lib.sh_compute.restype = _ci
lib.sh_plan_destroy.argtypes = [_vp]
lib.sh_plan_destroy.restype = None
lib.sh_last_error.argtypes = []
lib.sh_last_error.restype = _ci
lib.sh_last_error_string.argtypes = []
lib.sh_last_error_string.restype = ctypes.c_char_p


class ShError(RuntimeError):
    pass


def _fail():
    raise ShError("libpyr (sh) error %d: %s" % (lib.sh_last_error(), lib.sh_last_error_string().decode()))


def _ptr(t, shape, name):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
            and tuple(t.shape) == tuple(shape)):
        raise ValueError("%s must be a contiguous float32 CUDA tensor of shape %s" % (name, tuple(shape)))
    return t.data_ptr()


class Plan:
    """Owner of one ``sh_plan`` (see include/sh.h)."""

    def __init__(self, N_pup: int, n_sub: int, F: int, spot_binning: int, batch: int):
        self._h = lib.sh_plan_create(int(N_pup), int(n_sub), int(F), int(spot_binning), int(batch))
        if not self._h:
            _fail()
        self.N_pup, self.n_sub, self.F, self.bs, self.batch = int(N_pup), int(n_sub), int(F), int(spot_binning), int(batch)
        self.n_pix = self.F // self.bs

    def destroy(self):
        if self._h:
            lib.sh_plan_destroy(self._h)
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

    def empty_outputs(self, spots=False, device="cuda"):
        B, n = self.batch, self.n_sub
        s = torch.empty((B, 2, n, n), dtype=torch.float32, device=device)
        f = torch.empty((B, n, n), dtype=torch.float32, device=device)
        sp = torch.empty((B, n, n, self.n_pix, self.n_pix), dtype=torch.float32, device=device) if spots else None
        return s, f, sp

    def compute(self, amp, phase, out_slopes, out_flux=None, out_spots=None, stream=None):
        B, P, n = self.batch, self.N_pup, self.n_sub
        st = (stream if stream is not None else torch.cuda.current_stream()).cuda_stream
        rc = lib.sh_compute(self._h, _ptr(amp, (B, P, P), "amp"), _ptr(phase, (B, P, P), "phase"),
                            _ptr(out_slopes, (B, 2, n, n), "out_slopes"), _ptr(out_flux, (B, n, n), "out_flux"),
                            _ptr(out_spots, (B, n, n, self.n_pix, self.n_pix), "out_spots"), st)
        if rc:
            _fail()
