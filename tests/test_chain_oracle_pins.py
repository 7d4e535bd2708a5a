"""Pins of oracle/chain_oracle.c (atmosphere propagation, CCD noise model, PupData, Modalrec: SURVEY.md 8(f) f3)
against what mathematics and published values fix -- never against the CUDA path.  All CPU."""
import math
import os

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ch():
    from oracle import chain_oracle
    chain_oracle.build()
    return chain_oracle


# ---------------------------------------------------------------- atmosphere

def screens(L, S, seed):
    return np.random.default_rng(seed).standard_normal((L, S, S)).astype(np.float32)


def test_atmo_integer_shift_is_a_cyclic_roll(ch):
    """Integer displacement (dy, dx): phase[y][x] = screen[(y + dy) mod S][(x + dx) mod S] exactly (pins the
    sign of the displacement, the axis order and the periodic wrap)."""
    L, S, P = 1, 16, 16
    scr = screens(L, S, 1)
    for dy, dx in [(0, 0), (3, 0), (0, 5), (-2, 7), (16, -16), (35, -21)]:
        out = ch.atmo(scr, [[[dy, dx]]], P)
        assert np.array_equal(out[0], np.roll(scr[0].astype(np.float64), (-dy, -dx), axis=(0, 1))), (dy, dx)


def test_atmo_ramp_and_midpoint(ch):
    """A linear ramp is reproduced exactly by bilinear interpolation away from the wrap; a half-pixel shift of
    any screen is the mean of the two neighbours."""
    S, P = 32, 8
    yy, xx = np.mgrid[0:S, 0:S]
    ramp = (0.25 * yy - 0.5 * xx).astype(np.float32)[None]
    out = ch.atmo(ramp, [[[2.3, 4.7]]], P)
    y, x = np.mgrid[0:P, 0:P]
    assert np.allclose(out[0], 0.25 * (y + 2.3) - 0.5 * (x + 4.7), atol=1e-12)
    scr = screens(1, S, 2)
    out = ch.atmo(scr, [[[0.0, 0.5]]], S)
    s = scr[0].astype(np.float64)
    assert np.allclose(out[0], 0.5 * (s + np.roll(s, -1, axis=1)), atol=1e-15)
    out = ch.atmo(scr, [[[0.5, 0.0]]], S)
    assert np.allclose(out[0], 0.5 * (s + np.roll(s, -1, axis=0)), atol=1e-15)


def test_atmo_brute_force_and_linearity(ch):
    """Independent NumPy restatement (floor / fractional weights with fancy indexing), several layers, weights,
    per-source shifts; a transposed shift pair must fail."""
    L, S, P, B = 3, 24, 10, 2
    scr = screens(L, S, 3)
    rng = np.random.default_rng(4)
    sh = rng.uniform(-40, 40, size=(B, L, 2))
    w = np.array([0.7, -1.3, 2.0])
    out = ch.atmo(scr, sh, P, weights=w)

    def brute(sh):
        ref = np.zeros((B, P, P))
        y, x = np.mgrid[0:P, 0:P].astype(np.float64)
        for b in range(B):
            for l in range(L):
                Y, X = y + sh[b, l, 0], x + sh[b, l, 1]
                i, j = np.floor(Y).astype(int), np.floor(X).astype(int)
                fy, fx = Y - i, X - j
                s = scr[l].astype(np.float64)
                g = lambda a, c: s[np.mod(a, S), np.mod(c, S)]
                ref[b] += w[l] * ((1 - fy) * (1 - fx) * g(i, j) + (1 - fy) * fx * g(i, j + 1)
                                  + fy * (1 - fx) * g(i + 1, j) + fy * fx * g(i + 1, j + 1))
        return ref
    assert np.allclose(out, brute(sh), atol=1e-12)
    assert not np.allclose(out, brute(sh[:, :, ::-1]), atol=1e-3)
    # a constant screen is invariant; the sum over layers is linear
    const = np.full((1, S, S), 2.5, dtype=np.float32)
    assert np.allclose(ch.atmo(const, [[[1.37, -9.2]]], P), 2.5, atol=1e-13)
    parts = sum(w[l] * ch.atmo(scr[l:l + 1], sh[:, l:l + 1], P) for l in range(L))
    assert np.allclose(out, parts, atol=1e-12)
    # periodicity: a shift by S is the identity
    assert np.allclose(ch.atmo(scr, sh + S, P, weights=w), out, atol=1e-10)


# ---------------------------------------------------------------- Philox and the float32 maps

def test_philox_known_answer_vectors(ch):
    """Published known-answer vectors of Philox4x32-10 (tests/golden/philox4x32_10_kat.txt)."""
    n = 0
    for line in open(os.path.join(ROOT, "tests", "golden", "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        assert list(ch.philox(w[0:4], w[4:6])) == w[6:10]
        n += 1
    assert n == 3


def test_philox_counter_and_key_sensitivity(ch):
    a = ch.philox([5, 0, 0, 0], [1, 0])
    assert not np.array_equal(a, ch.philox([6, 0, 0, 0], [1, 0]))
    assert not np.array_equal(a, ch.philox([5, 1, 0, 0], [1, 0]))
    assert not np.array_equal(a, ch.philox([5, 0, 0, 0], [1, 1]))
    # equidistribution of the words over many counters: mean of u01 = 1/2, variance 1/12
    u = np.array([[ch.u01(w) for w in ch.philox([i, 7, 0, 0], [42, 0])] for i in range(4000)])
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.05


def test_u01_is_exact_and_open(ch):
    assert ch.u01(0) == 2.0 ** -24 and ch.u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert ch.u01(0x80000000) == 0.5 + 2.0 ** -24
    assert ch.u01(0x12345678) == ((0x12345678 >> 9) + 0.5) / 2 ** 23


def test_float_maps_against_libm(ch):
    """exp, log, cos(2 pi u) of the noise model are float32 polynomials; their values are pinned to libm."""
    rng = np.random.default_rng(0)
    for lam in list(rng.uniform(0, 30, 300)) + [0.0, 1e-6, 0.5, 29.999, 30.0, 79.0]:
        lam = float(np.float32(lam))
        assert abs(ch.exp_neg(lam) - math.exp(-lam)) <= 3e-7 * math.exp(-lam), lam
    for u in list(rng.uniform(0, 1, 300)) + [2.0 ** -24, 0.5, 0.70710678, 0.7071068, 1 - 2.0 ** -24, 1.0]:
        u = float(np.float32(u))
        assert abs(ch.log(u) - math.log(u)) <= 2e-7 * max(1.0, abs(math.log(u))), u
    for u in list(rng.uniform(0, 1, 400)) + [0.0, 0.125, 0.25, 0.375, 0.5, 0.625, 0.75, 0.875, 1 - 2.0 ** -24]:
        u = float(np.float32(u))
        assert abs(ch.cos2pi(u) - math.cos(2 * math.pi * u)) <= 3e-7, u


def test_normal_is_box_muller_and_standard(ch):
    rng = np.random.default_rng(1)
    ua, ub = rng.uniform(0, 1, 20000).astype(np.float32), rng.uniform(0, 1, 20000).astype(np.float32)
    z = np.array([ch.normal(a, b) for a, b in zip(ua, ub)])
    ref = np.sqrt(-2 * np.log(ua.astype(np.float64))) * np.cos(2 * np.pi * ub.astype(np.float64))
    assert np.abs(z - ref).max() <= 2e-6
    assert abs(z.mean()) < 0.03 and abs(z.var() - 1) < 0.04
    assert abs((z ** 3).mean()) < 0.1 and abs((z ** 4).mean() - 3) < 0.25


def test_poisson_inversion_is_the_quantile_function(ch):
    """lam < 30: the count is the Poisson quantile of ua (scipy), except where ua lies within the float32
    rounding of a CDF step."""
    from scipy import stats
    rng = np.random.default_rng(2)
    for lam in [0.01, 0.3, 1.0, 4.5, 12.0, 29.9]:
        lam32 = float(np.float32(lam))
        ua = rng.uniform(0, 1, 400).astype(np.float32)
        for u in ua:
            n = ch.poisson(lam32, float(u), 0.5)
            q = stats.poisson.ppf(float(u), lam32)
            if n != q:
                cdf = stats.poisson.cdf([min(n, q)], lam32)[0]
                assert abs(cdf - float(u)) < 3e-6 and abs(n - q) == 1, (lam, u, n, q)
    assert ch.poisson(0.0, 0.3, 0.3) == 0 and ch.poisson(-1.0, 0.3, 0.3) == 0
    assert ch.poisson(5.0, 2.0 ** -24, 0.1) == 0          # the smallest uniform gives the smallest count


def test_poisson_moments_both_branches(ch):
    rng = np.random.default_rng(3)
    for lam in [0.2, 3.0, 25.0, 30.0, 100.0, 5000.0]:
        ua, ub = rng.uniform(0, 1, 20000).astype(np.float32), rng.uniform(0, 1, 20000).astype(np.float32)
        n = np.array([ch.poisson(lam, a, b) for a, b in zip(ua, ub)])
        assert np.all(n == np.rint(n)) and n.min() >= 0
        assert abs(n.mean() - lam) < 4 * math.sqrt(lam / 20000) + 1e-3, lam
        assert abs(n.var() - lam) < 0.06 * lam + 0.01, lam


# ---------------------------------------------------------------- CCD

def test_ccd_noise_free_is_the_integral(ch):
    rng = np.random.default_rng(4)
    D = rng.uniform(0, 3, (2, 6, 6)).astype(np.float32)
    ccd = ch.CCD(D.shape, n_int=3, photon_noise=False, readout_noise=False)
    assert ccd.integrate(D, 2.0) is None and ccd.integrate(2 * D, 2.0) is None
    out = ccd.integrate(D, 4.0)
    assert np.allclose(out, 2 * D + 4 * D + 4 * D, rtol=1e-6)
    assert np.all(ccd.acc == 0)                     # cleared for the next frame
    # ADC: divide, round to nearest, clamp to [0, 2^bits - 1]
    ccd = ch.CCD((4,), n_int=1, photon_noise=False, readout_noise=False, adu_gain=2.0, n_bits=4)
    out = ccd.integrate(np.array([0.9, 5.0, 7.1, 100.0], dtype=np.float32), 1.0)
    assert list(out) == [0.0, 2.0, 4.0, 15.0]       # 0.45 -> 0, 2.5 -> 2 (ties to even), 3.55 -> 4, clamp 15


def test_ccd_noise_statistics_and_counters(ch):
    """Photon noise has mean = variance = the expected electrons; readout noise adds sigma^2; the draw depends
    on (pixel, frame, seed) only."""
    n = 40000
    lam = np.full(n, 12.0, dtype=np.float32)
    ccd = ch.CCD((n,), photon_noise=True, readout_noise=False, seed=9)
    f0, f1 = ccd.integrate(lam, 1.0), ccd.integrate(lam, 1.0)
    assert abs(f0.mean() - 12) < 0.08 and abs(f0.var() - 12) < 0.4
    assert not np.array_equal(f0, f1)               # next frame index: new draws
    again = ch.CCD((n,), photon_noise=True, readout_noise=False, seed=9).integrate(lam, 1.0)
    assert np.array_equal(f0, again)                # same (pixel, frame, seed): same draws
    other = ch.CCD((n,), photon_noise=True, readout_noise=False, seed=10).integrate(lam, 1.0)
    assert not np.array_equal(f0, other)
    ro = ch.CCD((n,), photon_noise=False, readout_noise=True, readout_level=2.0, seed=9).integrate(lam, 1.0)
    assert abs(ro.mean() - 12) < 0.05 and abs(ro.var() - 4) < 0.15
    both = ch.CCD((n,), photon_noise=True, readout_noise=True, readout_level=2.0, seed=9).integrate(lam, 1.0)
    assert abs(both.var() - 16) < 0.6
    assert abs(np.corrcoef(f0 - 12, both - f0)[0, 1]) < 0.03      # readout draw independent of the photon draw
    # the per-pixel model is the exported scalar functions on Philox words 0..3
    w = ch.philox([123, 0, 0, 0], [9, 0])
    e = ch.poisson(12.0, ch.u01(w[0]), ch.u01(w[1]))
    assert f0[123] == e
    assert both[123] == np.float32(np.float32(2.0) * np.float32(ch.normal(ch.u01(w[2]), ch.u01(w[3]))) + np.float32(e))


# ---------------------------------------------------------------- PupData, Modalrec

def test_pupdata_threshold(ch):
    Nd = 8
    ref = np.zeros((Nd, Nd), dtype=np.float32)
    ref[1, 1], ref[1, 5], ref[5, 1], ref[5, 5] = 1, 2, 3, 4          # same (Y, X) = (1, 1) in the four quadrants: T = 10
    ref[2, 3] = 2.9                                                     # (2, 3): T = 2.9
    ref[0, 6] = 3.0                                                     # quadrant b, (0, 2): T = 3.0
    v = ch.pupdata(ref, 0.3)
    assert v.shape == (4, 4) and v[1, 1] == 1 and v[2, 3] == 0 and v[0, 2] == 1 and v.sum() == 2
    assert ch.pupdata(ref, 0.0).sum() == 16


def test_modalrec_definition(ch):
    rng = np.random.default_rng(5)
    Nq, B, n_modes = 6, 3, 5
    valid = (rng.random((Nq, Nq)) < 0.6).astype(np.uint8)
    nv = int(valid.sum())
    s = rng.standard_normal((B, 2, Nq, Nq)).astype(np.float32)
    R = rng.standard_normal((n_modes, 2 * nv)).astype(np.float32)
    sv = np.concatenate([s[:, 0][:, valid.astype(bool)], s[:, 1][:, valid.astype(bool)]], axis=1).astype(np.float64)
    assert np.allclose(ch.modalrec(R, valid, s), sv @ R.astype(np.float64).T, atol=1e-12)
    # identity reconstructor: the compacted slope vector itself, sx first then sy, row-major over valid pixels
    assert np.array_equal(ch.modalrec(np.eye(2 * nv, dtype=np.float32), valid, s), sv)
    # a one-hot row picks one slope: the first valid pixel's sy is entry nv
    onehot = np.zeros((1, 2 * nv), dtype=np.float32)
    onehot[0, nv] = 1
    Y, X = np.argwhere(valid)[0]
    assert np.array_equal(ch.modalrec(onehot, valid, s)[:, 0], s[:, 1, Y, X].astype(np.float64))
