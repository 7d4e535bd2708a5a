"""Pins of the Shack-Hartmann oracle (oracle/sh_oracle.c) against what the mathematics fixes: a library
FFT of the zero-padded patch, brute force, Parseval, flat-wavefront symmetry, the exact cyclic shift of
the spot under an integer tilt, the sign and near-linearity of the centroid in a small tilt, validity
and the detector binning."""
import numpy as np
import pytest

TWO_PI = 2 * np.pi


@pytest.fixture(scope="module")
def sh():
    from oracle import sh_oracle
    sh_oracle.build()
    return sh_oracle


def cfreq(F):
    u = np.arange(F)
    return np.where(u < F // 2, u, u - F)


@pytest.mark.parametrize("p,F", [(4, 8), (6, 16), (8, 32), (5, 12)])
def test_spot_matches_library_fft(sh, p, F):
    rng = np.random.default_rng(p * F)
    e = rng.standard_normal((p, p)) + 1j * rng.standard_normal((p, p))
    z = np.zeros((F, F), complex)
    z[:p, :p] = e
    ref = np.abs(np.fft.fft2(z)) ** 2 / F ** 2
    assert np.allclose(sh.spot(e, F), ref, rtol=1e-12, atol=1e-12 * ref.max())


def test_spot_brute_force_and_orientation(sh):
    p, F = 3, 8
    rng = np.random.default_rng(1)
    e = rng.standard_normal((p, p)) + 1j * rng.standard_normal((p, p))
    S = np.zeros((F, F))
    for v in range(F):
        for u in range(F):
            acc = 0
            for y in range(p):
                for x in range(p):
                    acc += e[y, x] * np.exp(-1j * TWO_PI * (u * x + v * y) / F)
            S[v, u] = abs(acc) ** 2 / F ** 2
    assert np.allclose(sh.spot(e, F), S, atol=1e-13)
    assert not np.allclose(sh.spot(e, F), S.T, atol=1e-3)     # [v][u] = [y-frequency][x-frequency]


def test_parseval_flat_symmetry_and_validity(sh):
    P, n_sub, F, bs = 24, 3, 16, 2
    p = P // n_sub
    rng = np.random.default_rng(2)
    amp = rng.uniform(0.6, 1.0, (1, P, P)).astype(np.float32)
    amp[0, :p, :p] = 0.0                          # one dark sub-aperture
    amp[0, :p, p:2 * p] *= (rng.random((p, p)) < 0.3)   # one below the 50 % illumination threshold
    phase = rng.standard_normal((1, P, P)).astype(np.float32)
    s, fl, sp = sh.compute(P, n_sub, F, bs, amp, phase, want_spots=True)
    a2 = (amp[0].astype(np.float64) ** 2).reshape(n_sub, p, n_sub, p).sum((1, 3))
    assert np.allclose(fl[0], a2, rtol=1e-12)                     # Parseval per sub-aperture
    assert np.allclose(sp[0].sum((2, 3)), fl[0], rtol=1e-12)      # binning preserves flux
    assert s[0, 0, 0, 0] == 0 and s[0, 1, 0, 0] == 0 and s[0, 0, 0, 1] == 0 and s[0, 1, 0, 1] == 0
    # flat wavefront, uniform amplitude: spot symmetric about the axis, slopes exactly 0
    s0, _, sp0 = sh.compute(P, n_sub, F, bs, np.ones((1, P, P), np.float32), np.zeros((1, P, P), np.float32),
                            want_spots=True)
    assert np.abs(s0).max() < 1e-13
    full = sh.spot(np.ones((p, p), complex), F)
    c = cfreq(F)
    assert np.allclose(full[(-c) % F][:, (-c) % F], full, atol=1e-12)   # S(-v, -u) = S(v, u)


def test_integer_tilt_shifts_the_spot_exactly(sh):
    p, F, sx, sy = 8, 32, 3, -5
    rng = np.random.default_rng(3)
    A = rng.uniform(0.5, 1.0, (p, p))
    phi = 0.3 * rng.standard_normal((p, p))
    yy, xx = np.mgrid[0:p, 0:p]
    S0 = sh.spot(A * np.exp(1j * phi), F)
    S1 = sh.spot(A * np.exp(1j * (phi + TWO_PI * (sx * xx + sy * yy) / F)), F)
    assert np.allclose(S1, np.roll(S0, (sy, sx), axis=(0, 1)), atol=1e-12)   # f(u - s): the spot moves by +s


def test_centroid_sign_and_linearity(sh):
    P, n_sub, F, bs = 16, 2, 64, 1
    yy, xx = np.mgrid[0:P, 0:P]
    amp = np.ones((1, P, P), np.float32)
    out = []
    for a in (0.5, 1.0, 2.0):                     # tilt in focal samples: phase = 2 pi a x / F
        ph = (TWO_PI * a * xx / F).astype(np.float32)[None]
        s, _, _ = sh.compute(P, n_sub, F, bs, amp, ph)
        assert np.abs(s[0, 1]).max() < 1e-6       # no y response (float32 phase rounding only)
        assert np.all(s[0, 0] > 0)                # +x tilt -> +sx
        out.append(s[0, 0].mean())
    # the sinc^2 tails clipped by the cyclic F x F window bias the plain centre of gravity low, but it is
    # monotone and close to linear for small tilts
    assert out[0] < out[1] < out[2]
    assert abs(out[1] / out[0] - 2.0) < 0.05 and abs(out[2] / out[1] - 2.0) < 0.1
    assert 0.5 < out[1] <= 1.0


def test_detector_binning_and_bad_arguments(sh):
    P, n_sub, F = 8, 2, 8
    rng = np.random.default_rng(4)
    amp = np.ones((1, P, P), np.float32)
    ph = rng.standard_normal((1, P, P)).astype(np.float32)
    _, _, sp1 = sh.compute(P, n_sub, F, 1, amp, ph, want_spots=True)
    _, _, sp2 = sh.compute(P, n_sub, F, 2, amp, ph, want_spots=True)
    assert np.allclose(sp1.reshape(1, 2, 2, 4, 2, 4, 2).sum((4, 6)), sp2, rtol=1e-13)
    e = (amp[0, :4, :4] * np.exp(1j * ph[0, :4, :4].astype(np.float64)))
    S = sh.spot(e, F)
    assert np.allclose(sp1[0, 0, 0], np.fft.fftshift(S), rtol=1e-13)       # centred image, U = c(u) + F/2
    with pytest.raises(ValueError):
        sh.compute(9, 2, 8, 1, np.ones((1, 9, 9), np.float32), np.zeros((1, 9, 9), np.float32))
    with pytest.raises(ValueError):
        sh.compute(8, 2, 8, 3, amp, ph)
