"""Pins of the CPU oracle against things other than itself.

Every expected value here comes from a closed form, an invariant, NumPy written from the
definition (brute force), or numpy.fft used through a *different* identity (shift theorem,
separable operator) -- never from the oracle or from the CUDA path.
"""
import numpy as np
import pytest

from paper_2602_06688_b200 import synth

TWO_PI = 2.0 * np.pi


def disk(P, eps=0.0):
    a = 2 * np.arange(P) - (P - 1)
    r2 = a[:, None] ** 2 + a[None, :] ** 2
    return ((r2 <= P * P) & (r2 >= (eps * P) ** 2)).astype(np.float32)


def smooth_phase(P, seed, rms=1.0):
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:P, 0:P] / P
    ph = sum(rng.normal() * np.cos(TWO_PI * (i * x + j * y) + rng.uniform(0, TWO_PI))
             for i in range(3) for j in range(3))
    ph = ph - ph.mean()
    return (ph * rms / ph.std()).astype(np.float32)


# ---------------------------------------------------------------- P2: 1-D closed forms

@pytest.mark.parametrize("n", [1, 2, 4, 8, 64, 256, 12, 15, 7, 49, 55, 60, 121, 660, 1600])
def test_p2_dft_closed_forms(oracle, n):
    for f in (oracle.fft1d, oracle.dft_direct):
        for sign in (-1, +1):
            # delta at 0 -> constant 1
            d = np.zeros(n, complex); d[0] = 1
            assert np.allclose(f(d, sign), np.ones(n), atol=1e-13)
            # constant -> n * delta
            e = np.zeros(n, complex); e[0] = n
            assert np.allclose(f(np.ones(n), sign), e, atol=1e-11)
            # delta at x0 -> exp(sign 2 pi i u x0 / n)
            x0 = n // 3
            d = np.zeros(n, complex); d[x0] = 1
            assert np.allclose(f(d, sign), np.exp(sign * 1j * TWO_PI * np.arange(n) * x0 / n), atol=1e-12)
            # complex exponential exp(2 pi i s x / n) -> n delta[u - s] for sign -, delta[u + s] for sign +
            s = (n // 4 + 1) % n
            z = np.exp(1j * TWO_PI * s * np.arange(n) / n)
            e = np.zeros(n, complex); e[(s if sign < 0 else -s) % n] = n
            assert np.allclose(f(z, sign), e, atol=1e-10 * max(n, 1))


@pytest.mark.parametrize("n,w", [(16, 5), (64, 9), (256, 32)])
def test_p2_boxcar_dirichlet(oracle, n, w):
    x = np.zeros(n, complex); x[:w] = 1
    u = np.arange(1, n)
    expect = np.empty(n, complex)
    expect[0] = w
    # sum_{x<w} e^{-2 pi i u x/n} = e^{-i pi u (w-1)/n} sin(pi u w/n) / sin(pi u/n)
    expect[1:] = np.exp(-1j * np.pi * u * (w - 1) / n) * np.sin(np.pi * u * w / n) / np.sin(np.pi * u / n)
    assert np.allclose(oracle.fft1d(x, -1), expect, atol=1e-11)


@pytest.mark.parametrize("n", [8, 128, 2048])
def test_fft_matches_library_and_direct(oracle, n):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    assert np.allclose(oracle.fft1d(x, -1), np.fft.fft(x), atol=1e-10)
    assert np.allclose(oracle.fft1d(x, +1), np.fft.ifft(x) * n, atol=1e-10)
    if n <= 128:
        assert np.allclose(oracle.dft_direct(x, -1), np.fft.fft(x), atol=1e-10)


@pytest.mark.parametrize("n", [3, 5, 6, 9, 11, 12, 20, 25, 45, 49, 60, 77, 97, 121, 132, 242, 660, 1001, 1600])
def test_mixed_radix_matches_direct_dft(oracle, n):
    """The mixed-radix line transform used when N is not a power of two (the paper's 660 = 2^2 3 5 11
    and 1600 = 2^6 5^2) against the direct O(n^2) sum pyro_dft_direct -- primes,
    prime powers, products of distinct and repeated primes -- and against the library as a cross-check.
    A non-symmetric input: a wrong twiddle index, digit order or sign fails."""
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    x[n // 3] += 5.0
    for sign in (-1, +1):
        a = oracle.fft1d(x, sign)
        ref = oracle.dft_direct(x, sign)
        assert np.abs(a - ref).max() <= 1e-13 * n * np.abs(ref).max()
        lib = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
        assert np.abs(a - lib).max() <= 1e-13 * n * np.abs(lib).max()


@pytest.mark.parametrize("n,w", [(12, 5), (60, 9), (660, 220), (1600, 400)])
def test_mixed_radix_boxcar_dirichlet(oracle, n, w):
    """Closed form at the paper's sizes: a boxcar of the pupil width -> the Dirichlet kernel."""
    x = np.zeros(n, complex); x[:w] = 1
    u = np.arange(1, n)
    expect = np.empty(n, complex)
    expect[0] = w
    expect[1:] = np.exp(-1j * np.pi * u * (w - 1) / n) * np.sin(np.pi * u * w / n) / np.sin(np.pi * u / n)
    assert np.allclose(oracle.fft1d(x, -1), expect, atol=1e-10)


@pytest.mark.parametrize("n", [6, 12, 20, 66])
def test_dft2d_any_size_matches_library(oracle, n):
    """The 2-D transform used when N is not a power of two (the paper's 660, 1600): rows then columns of
    the mixed-radix line transform; also against the direct DFT applied along both axes."""
    rng = np.random.default_rng(n)
    x = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    assert np.allclose(oracle.fft2d(x, -1), np.fft.fft2(x), atol=1e-10 * n)
    assert np.allclose(oracle.fft2d(x, +1), np.fft.ifft2(x) * n * n, atol=1e-10 * n)
    rows = np.stack([oracle.dft_direct(r, -1) for r in x])
    both = np.stack([oracle.dft_direct(c, -1) for c in rows.T]).T
    assert np.allclose(oracle.fft2d(x, -1), both, atol=1e-10 * n)


def test_fft2d_matches_library(oracle):
    rng = np.random.default_rng(5)
    x = rng.normal(size=(32, 32)) + 1j * rng.normal(size=(32, 32))
    assert np.allclose(oracle.fft2d(x, -1), np.fft.fft2(x), atol=1e-10)
    assert np.allclose(oracle.fft2d(x, +1), np.fft.ifft2(x) * 32 * 32, atol=1e-10)
    # index order [v][u] = [y-frequency][x-frequency]: a pure x-wave lands in row 0
    yy, xx = np.mgrid[0:32, 0:32]
    F = oracle.fft2d(np.exp(1j * TWO_PI * 3 * xx / 32), -1)
    e = np.zeros((32, 32), complex); e[0, 3] = 32 * 32
    assert np.allclose(F, e, atol=1e-9)


# ---------------------------------------------------------------- P1: brute force O(N^4)

def brute_force_intensity(A, phi, N, M, r, mask=None, points=None):
    """The definition, literally: four-index sums with explicit complex exponentials."""
    P = A.shape[0]
    o = (N - P) // 2
    cp = (P - 1) / 2
    n = np.arange(N)
    f = np.where(n < N // 2, n, n - N)
    d = N // 4
    if mask is None:
        mask = np.exp(-1j * TWO_PI * d * (np.abs(f)[:, None] + np.abs(f)[None, :]) / N)   # [v][u]
    K = np.exp(-1j * TWO_PI * np.outer(n, n) / N)       # K[u][x]
    I = np.zeros((N, N))
    yy, xx = np.mgrid[0:P, 0:P]
    for k in range(M):
        th = TWO_PI * k / M
        ax, ay, wgt = r * np.cos(th), r * np.sin(th), 1.0
        if points is not None:
            ax, ay, wgt = points[0][k], points[1][k], points[2][k]
        E = np.zeros((N, N), complex)
        E[o:o + P, o:o + P] = A * np.exp(1j * (phi + (TWO_PI / P) * (ax * (xx - cp) + ay * (yy - cp))))
        F = np.einsum("vy,ux,yx->vu", K, K, E)           # sum_{y,x} E e^{-2 pi i (ux+vy)/N}
        G = F * mask
        O = np.einsum("vy,ux,vu->yx", K.conj(), K.conj(), G) / (N * N)
        I += wgt * np.abs(O) ** 2
    return I


@pytest.mark.parametrize("P,N,M,r", [(4, 8, 4, 1.0), (8, 16, 4, 1.5), (4, 16, 3, 0.7), (8, 32, 8, 2.0),
                                     (4, 12, 3, 1.0), (6, 20, 4, 1.5), (8, 24, 4, 2.0)])   # the last three: N not a power of two
def test_p1_brute_force(oracle, P, N, M, r):
    A = disk(P)
    A[0, 1] = 0.5   # break symmetry, non-binary amplitude
    phi = smooth_phase(P, 11 + N, 1.3)
    _, _, I = oracle.compute(P, N, M, r, 1, A, phi, want_full=True, nthreads=2)
    ref = brute_force_intensity(A.astype(float), phi.astype(float), N, M, r)
    assert np.max(np.abs(I[0] - ref)) <= 1e-12 * ref.max()


@pytest.mark.parametrize("P,N,M,r", [(4, 8, 4, 1.0), (8, 16, 3, 1.5)])
def test_p1_brute_force_general_mask(oracle, P, N, M, r):
    """The oracle's `mask` argument (what pyr_plan_set_mask is checked against): an arbitrary
    complex mask[v][u] -- amplitude and phase, neither separable nor symmetric, so a transposed
    or conjugated mask fails -- against the literal four-index sums."""
    rng = np.random.default_rng(5 + N)
    mask = (0.3 + rng.random((N, N))) * np.exp(1j * TWO_PI * rng.random((N, N)))
    A = disk(P)
    A[1, 0] = 0.4
    phi = smooth_phase(P, 23 + N, 1.1)
    _, _, I = oracle.compute(P, N, M, r, 1, A, phi, mask=mask, want_full=True, nthreads=2)
    ref = brute_force_intensity(A.astype(float), phi.astype(float), N, M, r, mask=mask)
    assert np.max(np.abs(I[0] - ref)) <= 1e-12 * ref.max()
    # and it is not accidentally insensitive to the orientation of the mask
    _, _, It = oracle.compute(P, N, M, r, 1, A, phi, mask=mask.T.copy(), want_full=True, nthreads=2)
    assert np.max(np.abs(It[0] - ref)) > 1e-3 * ref.max()


def test_points_entry(oracle):
    """pyr_oracle_compute_points (arbitrary modulation points and weights): brute force, the circle as a
    special case, Parseval with weights (sum D = sum_k w_k sum A^2), zero weights and repeated points."""
    P, N, M, b = 8, 16, 5, 2
    rng = np.random.default_rng(99)
    ax, ay, w = rng.uniform(-2, 2, M), rng.uniform(-2, 2, M), rng.uniform(0.2, 2.0, M)
    ay[3] = ay[1]                      # two points share a y-tilt
    A = disk(P)
    A[2, 1] = 0.6
    phi = smooth_phase(P, 31, 1.2)
    D, _, I = oracle.compute(P, N, M, 0.0, b, A, phi, want_full=True, nthreads=2, points=(ax, ay, w))
    ref = brute_force_intensity(A.astype(float), phi.astype(float), N, M, 0.0, points=(ax, ay, w))
    assert np.max(np.abs(I[0] - ref)) <= 1e-12 * ref.max()
    assert abs(D.sum() - w.sum() * (A.astype(float) ** 2).sum()) <= 1e-11 * D.sum()
    # the circle through the points entry
    th = TWO_PI * np.arange(8) / 8
    D0, s0, _ = oracle.compute(P, N, 8, 1.5, b, A, phi)
    D1, s1, _ = oracle.compute(P, N, 8, 0.0, b, A, phi, points=(1.5 * np.cos(th), 1.5 * np.sin(th), None))
    assert np.allclose(D0, D1, rtol=0, atol=1e-13 * D0.max()) and np.allclose(s0, s1, atol=1e-12)
    # a zero-weight point adds nothing; a repeated point is a doubled weight
    w0 = w.copy(); w0[2] = 0.0
    Dz, _, _ = oracle.compute(P, N, M, 0.0, b, A, phi, points=(ax, ay, w0))
    keep = [0, 1, 3, 4]
    Dk, _, _ = oracle.compute(P, N, 4, 0.0, b, A, phi, points=(ax[keep], ay[keep], w[keep]))
    assert np.allclose(Dz, Dk, rtol=0, atol=1e-13 * Dz.max())
    Dd, _, _ = oracle.compute(P, N, M + 1, 0.0, b, A, phi, points=(np.append(ax, ax[0]), np.append(ay, ay[0]), np.append(w, w[0])))
    w2 = w.copy(); w2[0] *= 2
    D2, _, _ = oracle.compute(P, N, M, 0.0, b, A, phi, points=(ax, ay, w2))
    assert np.allclose(Dd, D2, rtol=0, atol=1e-12 * D2.max())


def test_mask_is_fourth_roots(oracle):
    for N in (8, 16, 64):
        n = np.arange(N)
        f = np.where(n < N // 2, n, n - N)
        expect = np.exp(-1j * TWO_PI * (N // 4) * (np.abs(f)[:, None] + np.abs(f)[None, :]) / N)
        assert np.allclose(oracle.pyramid_mask(N), expect, atol=1e-12)


# ---------------------------------------------------------------- P3: Parseval

@pytest.mark.parametrize("P,N,M,r,b", [(16, 64, 8, 3.0, 2), (12, 32, 5, 1.3, 4), (32, 128, 8, 3.0, 2),
                                       (20, 60, 4, 3.0, 5), (22, 132, 3, 2.0, 11)])   # N = 60, 132 = 660/5: not powers of two
def test_p3_parseval(oracle, P, N, M, r, b):
    rng = np.random.default_rng(3)
    A = (disk(P, 0.3) * rng.uniform(0.5, 1.5, (P, P))).astype(np.float32)
    phi = smooth_phase(P, 7, 2.0)
    D, _, I = oracle.compute(P, N, M, r, b, A, phi, want_full=True)
    flux = M * np.sum(A.astype(float) ** 2)
    assert abs(I.sum() - flux) <= 1e-12 * flux
    assert abs(D.sum() - flux) <= 1e-12 * flux
    # and for an arbitrary pure-phase mask
    mk = np.exp(1j * rng.uniform(0, TWO_PI, (N, N)))
    D2, _, _ = oracle.compute(P, N, M, r, b, A, phi, mask=mk)
    assert abs(D2.sum() - flux) <= 1e-12 * flux


# ---------------------------------------------------------------- P4 / P5: identity and shift masks

def test_p4_identity_mask(oracle):
    P, N, M = 16, 64, 6
    A = disk(P, 0.25) * np.linspace(0.5, 1.0, P, dtype=np.float32)[None, :]
    phi = smooth_phase(P, 2, 3.0)
    _, _, I = oracle.compute(P, N, M, 2.5, 1, A, phi, mask=np.ones((N, N), complex), want_full=True)
    o = (N - P) // 2
    expect = np.zeros((N, N))
    expect[o:o + P, o:o + P] = M * A.astype(float) ** 2     # un-flipped (A is asymmetric in x)
    assert np.max(np.abs(I[0] - expect)) <= 1e-12


@pytest.mark.parametrize("dx,dy", [(5, 0), (0, 7), (-3, 11)])
def test_p5_shift_mask(oracle, dx, dy):
    P, N, M = 16, 64, 4
    A = disk(P) * np.linspace(0.5, 1.0, P, dtype=np.float32)[:, None]
    phi = smooth_phase(P, 4, 1.0)
    n = np.arange(N)
    mk = np.exp(-1j * TWO_PI * (dx * n[None, :] + dy * n[:, None]) / N)   # [v][u]
    _, _, I = oracle.compute(P, N, M, 1.0, 1, A, phi, mask=mk, want_full=True)
    o = (N - P) // 2
    base = np.zeros((N, N))
    base[o:o + P, o:o + P] = M * A.astype(float) ** 2
    expect = np.roll(base, (dy, dx), axis=(0, 1))          # shifted by (+dx, +dy)
    assert np.max(np.abs(I[0] - expect)) <= 1e-12


# ---------------------------------------------------------------- P6: flat wavefront

@pytest.mark.parametrize("P,N,M,r,b,eps", [(16, 64, 8, 3.0, 2, 0.0), (24, 128, 12, 2.0, 2, 0.3),
                                           (20, 60, 8, 3.0, 5, 0.0)])   # N = 60: not a power of two
def test_p6_flat_wavefront(oracle, P, N, M, r, b, eps):
    A = disk(P, eps)
    phi = np.zeros((P, P), np.float32)
    D, S, I = oracle.compute(P, N, M, r, b, A, phi, want_full=True)
    I = I[0]; D = D[0]
    assert np.max(np.abs(I - I[:, ::-1])) <= 1e-13 * I.max()
    assert np.max(np.abs(I - I[::-1, :])) <= 1e-13 * I.max()
    Nq = N // b // 2
    q = [D[:Nq, :Nq].sum(), D[:Nq, Nq:].sum(), D[Nq:, :Nq].sum(), D[Nq:, Nq:].sum()]
    flux = M * np.sum(A.astype(float) ** 2)
    assert np.allclose(q, flux / 4, rtol=1e-12)
    assert np.max(np.abs(S)) <= 1e-13
    # the four pupil images are translates of each other
    assert np.allclose(D[:Nq, :Nq], D[:Nq, Nq:][:, ::-1], atol=1e-13 * D.max())


# ---------------------------------------------------------------- P7: slope sign, linearity

def test_p7_tilt_sign_and_linearity(oracle):
    P, N, M, r, b = 40, 128, 24, 3.0, 2
    A = disk(P)
    yy, xx = np.mgrid[0:P, 0:P]
    cp = (P - 1) / 2
    valid = synth.valid_from_amplitude(A, N, b)
    means = []
    for alpha in (0.02, 0.04, 0.08):
        phi = (alpha * TWO_PI * (xx - cp) / P).astype(np.float32)
        _, S, _ = oracle.compute(P, N, M, r, b, A, phi, valid=valid)
        v = valid.astype(bool)
        sx, sy = S[0, 0][v].mean(), S[0, 1][v].mean()
        assert sx > 0, "positive x tilt must give positive sx (reading S8)"
        assert abs(sy) <= 1e-6 * sx
        means.append(sx / alpha)
    assert np.allclose(means, means[0], rtol=2e-3), means     # linear for alpha << r
    # y tilt -> sy, same gain
    phi = (0.04 * TWO_PI * (yy - cp) / P).astype(np.float32)
    _, S, _ = oracle.compute(P, N, M, r, b, A, phi, valid=valid)
    v = valid.astype(bool)
    assert np.isclose(S[0, 1][v].mean() / 0.04, means[1], rtol=1e-5)
    assert abs(S[0, 0][v].mean()) <= 1e-6 * S[0, 1][v].mean()


def test_p12_geometric_gain_soft(oracle):
    """Soft sanity, not parity: sx ~ (2/pi) asin(alpha/r) within ~25 % for M >= 24."""
    P, N, M, r, b = 80, 256, 24, 3.0, 2
    A = disk(P)
    yy, xx = np.mgrid[0:P, 0:P]
    alpha = 0.5
    phi = (alpha * TWO_PI * (xx - (P - 1) / 2) / P).astype(np.float32)
    valid = synth.valid_from_amplitude(A, N, b)
    _, S, _ = oracle.compute(P, N, M, r, b, A, phi, valid=valid)
    sx = S[0, 0][valid.astype(bool)].mean()
    geo = (2 / np.pi) * np.arcsin(alpha / r)
    assert 0.9 * geo < sx < 1.3 * geo, (sx, geo)


# ---------------------------------------------------------------- P8: translation equivariance

def test_p8_translation(oracle):
    P, N, M, r = 24, 64, 8, 2.0
    A = np.zeros((P, P), np.float32)
    A[6:18, 6:18] = disk(12) * np.linspace(0.6, 1.0, 12, dtype=np.float32)[None, :]
    phi = np.zeros((P, P), np.float32)
    phi[6:18, 6:18] = smooth_phase(12, 9, 1.5)
    _, _, I0 = oracle.compute(P, N, M, r, 1, A, phi, want_full=True)
    for sy, sx in [(3, 0), (0, -4), (5, 2), (-6, 6)]:
        A2 = np.roll(A, (sy, sx), axis=(0, 1))
        p2 = np.roll(phi, (sy, sx), axis=(0, 1))
        _, _, I2 = oracle.compute(P, N, M, r, 1, A2, p2, want_full=True)
        assert np.max(np.abs(I2[0] - np.roll(I0[0], (sy, sx), axis=(0, 1)))) <= 1e-12 * I0.max()


# ---------------------------------------------------------------- P9: dihedral equivariance

def test_p9_dihedral(oracle):
    P, N, M, r, b = 16, 64, 8, 2.0, 2
    A = disk(P, 0.2) * np.linspace(0.6, 1.0, P, dtype=np.float32)[None, :]
    phi = smooth_phase(P, 21, 1.2)
    valid = synth.valid_from_amplitude(disk(P, 0.2), N, b)
    D, S, _ = oracle.compute(P, N, M, r, b, A, phi, valid=valid)
    # transpose
    Dt, St, _ = oracle.compute(P, N, M, r, b, A.T.copy(), phi.T.copy(), valid=valid.T.copy())
    assert np.max(np.abs(Dt[0] - D[0].T)) <= 1e-12 * D.max()
    assert np.max(np.abs(St[0, 0] - S[0, 1].T)) <= 1e-12
    assert np.max(np.abs(St[0, 1] - S[0, 0].T)) <= 1e-12
    # flip x
    Df, Sf, _ = oracle.compute(P, N, M, r, b, A[:, ::-1].copy(), phi[:, ::-1].copy(), valid=valid[:, ::-1].copy())
    assert np.max(np.abs(Df[0] - D[0][:, ::-1])) <= 1e-12 * D.max()
    assert np.max(np.abs(Sf[0, 0] + S[0, 0][:, ::-1])) <= 1e-12
    assert np.max(np.abs(Sf[0, 1] - S[0, 1][:, ::-1])) <= 1e-12


# ---------------------------------------------------------------- P10: tilt scale via shift theorem

@pytest.mark.parametrize("k_of_4", [0, 1, 2, 3])
def test_p10_integer_focal_shift(oracle, k_of_4):
    """A tilt of a lambda/D moves the focal-plane field by a*N/P samples.  With M=4 the four
    points are (+x, +y, -x, -y); build the expected sum from numpy.fft + np.roll."""
    P, N, r = 32, 128, 3.0          # s = r N / P = 12 samples (config C1 geometry)
    s = int(round(r * N / P))
    A = synth.pupil_amplitude(P, 0)
    phi = smooth_phase(P, 5, 1.0)
    o = (N - P) // 2
    E0 = np.zeros((N, N), complex)
    E0[o:o + P, o:o + P] = A * np.exp(1j * phi.astype(float))
    F0 = np.fft.fft2(E0)
    n = np.arange(N)
    f = np.where(n < N // 2, n, n - N)
    mask = (-1j) ** ((np.abs(f)[:, None] + np.abs(f)[None, :]) % 4)
    shifts = [(0, s), (s, 0), (0, -s), (-s, 0)]            # (dv, du) for k = 0..3
    expect = np.zeros((N, N))
    for dv, du in shifts:
        expect += np.abs(np.fft.ifft2(np.roll(F0, (dv, du), axis=(0, 1)) * mask)) ** 2
    _, _, I = oracle.compute(P, N, 4, r, 1, A, phi, want_full=True)
    assert np.max(np.abs(I[0] - expect)) <= 1e-11 * expect.max()
    # and a single point (M=1 -> theta=0 -> +x)
    _, _, I1 = oracle.compute(P, N, 1, r, 1, A, phi, want_full=True)
    e1 = np.abs(np.fft.ifft2(np.roll(F0, (0, s), axis=(0, 1)) * mask)) ** 2
    assert np.max(np.abs(I1[0] - e1)) <= 1e-11 * e1.max()


# ---------------------------------------------------------------- P11: separable operator

def test_p11_separable_identity(oracle):
    P, N, M, r = 16, 64, 8, 2.5
    A = disk(P, 0.2)
    phi = smooth_phase(P, 8, 2.0)
    n = np.arange(N)
    f = np.where(n < N // 2, n, n - N)
    g = (-1j) ** (np.abs(f) % 4)
    C = np.fft.ifft(g[:, None] * np.fft.fft(np.eye(N), axis=0), axis=0)    # F^-1 diag(g) F
    o = (N - P) // 2
    cp = (P - 1) / 2
    yy, xx = np.mgrid[0:P, 0:P]
    expect = np.zeros((N, N))
    for k in range(M):
        th = TWO_PI * k / M
        E = np.zeros((N, N), complex)
        E[o:o + P, o:o + P] = A * np.exp(1j * (phi + TWO_PI / P * r * (np.cos(th) * (xx - cp) + np.sin(th) * (yy - cp))))
        expect += np.abs(C @ E @ C.T) ** 2
    _, _, I = oracle.compute(P, N, M, r, 1, A, phi, want_full=True)
    assert np.max(np.abs(I[0] - expect)) <= 1e-12 * expect.max()


# ---------------------------------------------------------------- rebin / slopes / validity

def test_rebin_and_slopes_definitions(oracle):
    rng = np.random.default_rng(0)
    N, b = 32, 4
    I = rng.uniform(size=(N, N))
    D = oracle.rebin(I, b)
    assert np.allclose(D, I.reshape(N // b, b, N // b, b).sum(axis=(1, 3)), rtol=1e-14)
    Nd = N // b; Nq = Nd // 2
    valid = (rng.uniform(size=(Nq, Nq)) > 0.3).astype(np.uint8)
    S = oracle.slopes_from_D(D, valid)
    Qa, Qb, Qc, Qd = D[:Nq, :Nq], D[:Nq, Nq:], D[Nq:, :Nq], D[Nq:, Nq:]
    v = valid.astype(bool)
    T = (Qa + Qb + Qc + Qd)[v].mean()
    assert np.allclose(S[0], np.where(v, ((Qb + Qd) - (Qa + Qc)) / T, 0), rtol=1e-13)
    assert np.allclose(S[1], np.where(v, ((Qc + Qd) - (Qa + Qb)) / T, 0), rtol=1e-13)


@pytest.mark.parametrize("P,N,b", [(32, 128, 2), (80, 256, 2), (160, 512, 4), (120, 512, 4), (480, 2048, 8),
                                   (220, 660, 5), (30, 120, 2), (36, 96, 4)])
def test_default_valid_is_the_geometric_pupil_image(oracle, P, N, b):
    """Pin of pyro_default_valid against the geometry, not its integer formula:
    a detector pixel is valid iff its CENTRE lies inside the circle of the pupil image, which is centred
    on the quadrant (N_q / 2 detector pixels from its corner) and n_s = P / b pixels across."""
    v = oracle.default_valid(P, N, b).astype(bool)
    Nq, ns = N // b // 2, P // b
    assert v.shape == (Nq, Nq)
    cy = np.arange(Nq) + 0.5 - Nq / 2.0                     # pixel centres relative to the image centre
    d = np.hypot(cy[:, None], cy[None, :])
    margin = np.abs(d - ns / 2.0)
    on_edge = margin < 1e-9                                 # centre exactly on the circle: counts as inside
    assert np.array_equal(v[~on_edge], (d < ns / 2.0)[~on_edge])
    assert np.all(v[on_edge])
    # the 8-fold symmetry of a centred circle on a centred grid
    assert np.array_equal(v, v[::-1, :]) and np.array_equal(v, v[:, ::-1]) and np.array_equal(v, v.T)
    # pixel count = area of the disc up to a boundary layer one pixel thick
    assert abs(int(v.sum()) - np.pi * ns * ns / 4.0) <= 2 * ns
    # fits inside the quadrant, touches the inscribed square's edge rows
    assert not v[0, 0] and v[Nq // 2, Nq // 2]
    assert v.any(axis=1).sum() == (ns if (ns - Nq) % 2 == 0 else ns - 1) or ns >= Nq


def test_thread_count_does_not_matter(oracle):
    c = synth.CONFIGS[1]
    amp, phase = synth.make_inputs(c)
    D1, S1, _ = oracle.compute(c.P, c.N, c.M, c.r, c.b, amp, phase, nthreads=1)
    D3, S3, _ = oracle.compute(c.P, c.N, c.M, c.r, c.b, amp, phase, nthreads=3)
    assert np.max(np.abs(D1 - D3)) <= 1e-13 * D1.max()
    assert np.max(np.abs(S1 - S3)) <= 1e-12


def test_bad_arguments(oracle):
    A = np.ones((1, 4, 4), np.float32)
    with pytest.raises(ValueError):
        oracle.compute(4, 13, 4, 1.0, 1, A, A)      # N odd
    with pytest.raises(ValueError):
        oracle.compute(4, 16, 0, 1.0, 1, A, A)      # M < 1


# ---------------------------------------------------------------- f4: PolyCromPyramid and ModulatedDoubleRoof

def brute_force_double_roof(A, phi, N, M, r, kappa):
    """Reading DR1, literally: DFT2, x-roof, inverse DFT2, pupil-plane quadratic phase, DFT2, y-roof, inverse DFT2."""
    P = A.shape[0]
    o, cp, c = (N - P) // 2, (P - 1) / 2, (N - 1) / 2
    n = np.arange(N)
    f = np.abs(np.where(n < N // 2, n, n - N))
    roof = np.exp(-1j * TWO_PI * (N // 4) * f / N)
    K = np.exp(-1j * TWO_PI * np.outer(n, n) / N)
    q = np.exp(1j * np.pi * kappa * ((n[None, :] - c) ** 2 + (n[:, None] - c) ** 2))     # [y][x]
    I = np.zeros((N, N))
    yy, xx = np.mgrid[0:P, 0:P]
    for k in range(M):
        th = TWO_PI * k / M
        E = np.zeros((N, N), complex)
        E[o:o + P, o:o + P] = A * np.exp(1j * (phi + (TWO_PI / P) * (r * np.cos(th) * (xx - cp) + r * np.sin(th) * (yy - cp))))
        F1 = np.einsum("vy,ux,yx->vu", K, K, E) * roof[None, :]                # roof 1: function of u (x-frequency)
        mid = np.einsum("vy,ux,vu->yx", K.conj(), K.conj(), F1) / (N * N) * q
        F2 = np.einsum("vy,ux,yx->vu", K, K, mid) * roof[:, None]              # roof 2: function of v
        O = np.einsum("vy,ux,vu->yx", K.conj(), K.conj(), F2) / (N * N)
        I += np.abs(O) ** 2
    return I


@pytest.mark.parametrize("P,N,M,r,kappa", [(4, 8, 4, 1.0, 0.02), (8, 16, 4, 1.5, 0.005), (6, 20, 3, 1.0, -0.01)])
def test_double_roof_brute_force(oracle, P, N, M, r, kappa):
    A = disk(P)
    A[0, 1] = 0.5
    phi = smooth_phase(P, 21, 1.0)
    _, _, I = oracle.compute(P, N, M, r, 1, A.astype(np.float32), phi, want_full=True, double_roof=kappa)
    ref = brute_force_double_roof(A.astype(np.float32).astype(np.float64), phi.astype(np.float64), N, M, r, kappa)
    assert np.abs(I[0] - ref).max() <= 1e-12 * ref.max()
    # swapping the two roofs' axes (transposed input and output) is NOT the same sensor when kappa != 0
    _, _, It = oracle.compute(P, N, M, r, 1, A.T.astype(np.float32).copy(), phi.T.copy(), want_full=True, double_roof=kappa)
    assert np.abs(It[0].T - ref).max() > 1e-6 * ref.max()


def test_double_roof_limits_and_identity(oracle):
    """kappa = 0: the two roofs multiply to the four-face pyramid.  Any kappa: unit-modulus factors, so Parseval
    holds; and the sensor equals the pyramid fed with the extra cylindrical phase pi kappa (y - c_p)^2 (the x part
    of q multiplies the output, the y part the input: DESIGN.md section 15)."""
    P, N, M, r, b = 16, 64, 8, 2.0, 2
    A = disk(P).astype(np.float32)
    phi = smooth_phase(P, 5, 1.5)
    D0, s0, _ = oracle.compute(P, N, M, r, b, A, phi)
    D1, s1, _ = oracle.compute(P, N, M, r, b, A, phi, double_roof=0.0)
    assert np.abs(D1 - D0).max() <= 1e-13 * D0.max() and np.abs(s1 - s0).max() <= 1e-12
    kappa = 0.004
    D2, s2, _ = oracle.compute(P, N, M, r, b, A, phi, double_roof=kappa)
    assert abs(D2.sum() - M * float((A.astype(np.float64) ** 2).sum())) <= 1e-11 * D2.sum()
    assert np.abs(D2 - D0).max() > 1e-3 * D0.max()
    y = np.arange(P) - (P - 1) / 2
    phi_c = (phi.astype(np.float64) + np.pi * kappa * (y ** 2)[:, None]).astype(np.float32)
    D3, s3, _ = oracle.compute(P, N, M, r, b, A, phi_c)
    assert np.abs(D3 - D2).max() <= 1e-6 * D2.max()        # float32 rounding of the modified phase only


def test_poly_brute_force_and_limits(oracle):
    P, N, M, r = 8, 16, 4, 1.5
    A = disk(P)
    A[0, 1] = 0.5
    phi = smooth_phase(P, 8, 1.2)
    A32, p64 = A.astype(np.float32), phi.astype(np.float64)
    ratio, weight = np.array([1.0, 0.8, 1.25]), np.array([0.5, 1.0, 0.25])
    _, _, I = oracle.compute(P, N, M, r, 1, A32, phi, want_full=True, poly=(ratio, weight))
    # every wavelength is the monochromatic definition with the whole pupil phase (turbulence and tilt) scaled
    ref = sum(w * brute_force_intensity(A32.astype(np.float64), s * p64, N, M, s * r) for s, w in zip(ratio, weight))
    assert np.abs(I[0] - ref).max() <= 1e-12 * ref.max()
    assert abs(I.sum() - weight.sum() * M * float((A32.astype(np.float64) ** 2).sum())) <= 1e-11 * I.sum()
    # one wavelength at ratio 1 is the monochromatic sensor; ratio 2 = phase and radius doubled (exact in float32)
    D0, s0, _ = oracle.compute(P, N, M, r, 2, A32, phi)
    D1, s1, _ = oracle.compute(P, N, M, r, 2, A32, phi, poly=([1.0], None))
    assert np.array_equal(D0, D1) and np.array_equal(s0, s1)
    D2, _, _ = oracle.compute(P, N, M, 2 * r, 2, A32, (2 * phi).astype(np.float32))
    D3, _, _ = oracle.compute(P, N, M, r, 2, A32, phi, poly=([2.0], None))
    assert np.abs(D2 - D3).max() <= 1e-13 * D2.max()
    with pytest.raises(ValueError):
        oracle.compute(P, N, M, r, 2, A32, phi, poly=([1.0, 0.9], [1.0, -1.0]))
