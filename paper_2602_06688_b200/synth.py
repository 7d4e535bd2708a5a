"""Seeded synthetic inputs for the five BASELINE.json workloads.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only makes pupil amplitudes, Kolmogorov-like phase screens and the
sub-aperture validity map handed to both sides.  Recipe: SURVEY.md section 8(d) / DESIGN.md
"Input recipe".  The paper's own inputs (SOUL / ANDES / MORFEO loops) need
calibration data that is not public; these shapes stand in for them.

Pure NumPy; imports nothing from the CUDA binding or from ``oracle/``.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    """One row of SURVEY.md section 8 config table."""
    cfg: int          # 1..5
    name: str
    P: int            # N_pup
    N: int            # N_fft
    M: int            # n_mod
    r: float          # modulation radius, lambda/D
    b: int            # binning
    B: int            # batch (sources per pyr_compute call)
    steps: int        # time steps of new phase per run
    eps_pct: int      # central obstruction, percent of diameter
    sigma: float      # phase rms over the pupil, rad

    @property
    def N_det(self) -> int:
        return self.N // self.b

    @property
    def N_q(self) -> int:
        return self.N // self.b // 2

    @property
    def nominal_flops_per_frame(self) -> float:
        """2*M 2-D FFTs x 5 N^2 log2(N^2) (BASELINE.json north_star)."""
        import math
        return 2.0 * self.M * 5.0 * self.N * self.N * math.log2(self.N * self.N)


CONFIGS = {
    1: Config(1, "C1-tiny", 32, 128, 8, 3.0, 2, 1, 1, 0, 1.0),
    2: Config(2, "C2-soul-like", 80, 256, 24, 3.0, 2, 1, 1, 0, 2.0),
    3: Config(3, "C3-timeseries", 160, 512, 48, 4.0, 4, 1, 16, 30, 3.0),
    4: Config(4, "C4-multisource", 120, 512, 36, 3.0, 4, 6, 1, 28, 2.5),
    5: Config(5, "C5-elt", 480, 2048, 64, 4.0, 8, 2, 1, 28, 4.0),
}

# The paper's own pyramid FFT workloads (Table 2; SOUL: 220 px pupil x
# oversampling 3, 40 sub-apertures, 24 modulation steps at 3 lambda/D, PAPER.md:410-414, 534, 609;
# ANDES: 400 px x 4, 24 steps), with synthetic seeded inputs as everywhere else.  Not among the
# five BASELINE.json configs; bench.py reports them as context (their N_fft is not a power of two).
PAPER_SHAPES = {
    "SOUL_24x660x660": Config(6, "soul-660", 220, 660, 24, 3.0, 5, 1, 1, 0, 2.0),
    "ANDES_24x1600x1600": Config(7, "andes-1600", 400, 1600, 24, 3.0, 8, 1, 1, 28, 3.0),
}


def pupil_amplitude(P: int, eps_pct: int) -> np.ndarray:
    """Binary annular pupil on a P x P grid, float32.  Integer arithmetic, no ties."""
    a = 2 * np.arange(P, dtype=np.int64) - (P - 1)
    r2 = a[:, None] ** 2 + a[None, :] ** 2
    inside = r2 <= P * P
    outside_obstruction = 10000 * r2 >= (eps_pct * eps_pct) * P * P
    return (inside & outside_obstruction).astype(np.float32)


def kolmogorov_phase(P: int, amp: np.ndarray, sigma: float, seed: int) -> np.ndarray:
    """White noise filtered by f^(-11/6) on a 2P grid, cropped to P x P, piston removed over
    the pupil and scaled to ``sigma`` rad rms over the pupil; zero outside; float32."""
    rng = np.random.Generator(np.random.PCG64(seed))
    w = rng.standard_normal((2 * P, 2 * P))
    W = np.fft.fft2(w)
    f = np.fft.fftfreq(2 * P) * (2 * P)
    ff = np.hypot(f[:, None], f[None, :])
    filt = np.zeros_like(ff)
    nz = ff > 0
    filt[nz] = ff[nz] ** (-11.0 / 6.0)
    s = np.real(np.fft.ifft2(W * filt))[:P, :P]
    m = amp > 0
    s = s - s[m].mean()
    s = s * (sigma / np.sqrt(np.mean(s[m] ** 2)))
    s = np.where(m, s, 0.0)
    return s.astype(np.float32)


def seed_for(cfg: int, source: int, step: int) -> int:
    return 1000 * cfg + 100 * source + step


def make_inputs(c: Config, step: int = 0):
    """(amp, phase) float32 arrays of shape [B][P][P] for time step ``step``."""
    A = pupil_amplitude(c.P, c.eps_pct)
    amp = np.repeat(A[None], c.B, axis=0).copy()
    phase = np.stack([kolmogorov_phase(c.P, A, c.sigma, seed_for(c.cfg, s, step)) for s in range(c.B)])
    return amp, phase


def valid_from_amplitude(A: np.ndarray, N: int, b: int) -> np.ndarray:
    """Sub-aperture validity map [N_q][N_q] (uint8) handed to both sides: a detector pixel
    of the pupil image is valid iff at least half of its b x b pupil samples are lit."""
    P = A.shape[0]
    Nq = N // b // 2
    ns = P // b
    q0 = (N // 4 - P // 2) // b
    lit = (A > 0).astype(np.int64).reshape(ns, b, ns, b).sum(axis=(1, 3))
    v = np.zeros((Nq, Nq), dtype=np.uint8)
    v[q0:q0 + ns, q0:q0 + ns] = (2 * lit >= b * b).astype(np.uint8)
    return v


# Shack-Hartmann workloads, Table 2's "n_subapertures x FFT x FFT" at the paper's own FFT
# sizes: (P, n_sub, F, spot_binning, batch, phase rms).  The lenslet counts follow the paper (314 ~ pi/4 20^2,
# 1256 ~ pi/4 40^2, 3630 ~ pi/4 68^2 lit sub-apertures, 6 LGS).  Pupil sampling: SCAO SH and ERIS use the paper's
# 160 px pupil (p = 8 and 4 px per lenslet); MORFEO's 480 px over 68 lenslets is not an integer, so the pupil is
# sampled at 544 = 68 x 8 px (reading SH1: an integer number of pixels per lenslet).  The spot binning is not
# printed; it is chosen to give 8 x 8, 4 x 4 and 16 x 16 detector pixels per sub-aperture.
SH_SHAPES = {
    "SH_SCAO_314x56x56": (160, 20, 56, 7, 1, 6.0),
    "SH_ERIS_1256x68x68": (160, 40, 68, 17, 1, 8.0),
    "SH_MORFEO_6x3630x240x240": (544, 68, 240, 15, 6, 10.0),
}


def make_sh_inputs(P: int, B: int, sigma: float, seed: int = 4242):
    A = pupil_amplitude(P, 28)
    amp = np.repeat(A[None], B, axis=0).copy()
    phase = np.stack([kolmogorov_phase(P, A, sigma, seed + s) for s in range(B)])
    return amp.astype(np.float32), phase.astype(np.float32)
