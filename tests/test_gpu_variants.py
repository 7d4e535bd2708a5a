"""GPU parity of the sensor variants of SURVEY.md 8(f) f4 against the oracle: PolyCromPyramid
(pyr_plan_create_poly) and ModulatedDoubleRoof (pyr_plan_set_double_roof); plus the
half-sample-apex convention of f1 as a custom separable mask.  north_star's tolerances throughout."""
import numpy as np
import pytest

from paper_2602_06688_b200 import synth

pytestmark = pytest.mark.gpu

TOL_MAX, TOL_L2, TOL_S = 1e-4, 1e-5, 1e-4


@pytest.fixture(scope="module")
def pyr():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2602_06688_b200 import build
    build.build()
    from paper_2602_06688_b200 import pyr as m
    return m


@pytest.fixture(scope="module")
def oracle():
    from oracle import pyr_oracle
    pyr_oracle.build()
    return pyr_oracle


def inputs(P, B, seed, sigma=1.5, eps=0):
    amp = np.stack([synth.pupil_amplitude(P, eps) for _ in range(B)])
    phase = np.stack([synth.kolmogorov_phase(P, amp[0], sigma, seed + s) for s in range(B)])
    return amp.astype(np.float32), phase.astype(np.float32)


def run(plan, amp, phase):
    import torch
    I, s = plan.empty_outputs()
    I.fill_(float("nan"))
    s.fill_(float("nan"))
    plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
    torch.cuda.synchronize()
    return I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)


def check(D, s, D_ref, s_ref):
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(s))
    dmax = np.abs(D - D_ref).max() / D_ref.max()
    l2 = np.linalg.norm((D - D_ref).ravel()) / np.linalg.norm(D_ref.ravel())
    ds = np.abs(s - s_ref).max()
    assert dmax <= TOL_MAX and l2 <= TOL_L2 and ds <= TOL_S, "%.3e %.3e %.3e" % (dmax, l2, ds)


POLY = [
    # P, N, M, r, b, B, ratios, weights
    (8, 32, 4, 1.5, 1, 1, [1.0, 0.8], None),
    (32, 128, 8, 3.0, 2, 2, [1.0, 0.85, 1.2], [0.5, 1.0, 0.25]),
    (80, 256, 24, 3.0, 2, 1, [0.9, 1.0, 1.1], None),                 # C2 shape, three wavelengths
    (120, 512, 12, 3.0, 4, 2, [1.0, 0.7], [1.0, 2.0]),
    (160, 1024, 6, 4.0, 8, 1, [1.0, 1.3], [0.3, 0.7]),
    (480, 2048, 8, 4.0, 8, 2, [0.9, 1.0, 1.1], [0.25, 0.5, 0.25]),     # C5 shape: k_field per wavelength + k_cols_t / k_rows_t
    (20, 60, 5, 3.0, 5, 1, [1.0, 0.8], None),                         # N_fft not a power of two, odd M (table kernels)
    (220, 660, 6, 3.0, 5, 1, [1.0, 0.9], [1.0, 0.5]),                 # SOUL size
    # ONE wavelength other than the reference one (a random sweep found the phase left unscaled for a single group)
    (32, 128, 3, 1.0, 16, 2, [0.8], [2.0]),
    (20, 60, 5, 3.0, 5, 1, [0.7345], None),                           # table kernels
    (192, 2048, 3, 2.0, 8, 1, [1.21], [0.5]),                         # k_field path
    (96, 1024, 2, 2.0, 4, 1, [0.9], None),
]


@pytest.mark.parametrize("P,N,M,r,b,B,ratio,weight", POLY)
def test_poly_parity(pyr, oracle, P, N, M, r, b, B, ratio, weight):
    big = P >= 120
    amp, phase = inputs(P, B, 700 + N, sigma=2.5 if big else 1.5, eps=28 if big else 0)
    with pyr.Plan(P, N, M, r, b, B, poly=(ratio, weight)) as plan:
        D, s = run(plan, amp, phase)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, poly=(np.float32(ratio).astype(np.float64),
                                                                   None if weight is None else np.float32(weight).astype(np.float64)))
    check(D, s, D_ref, s_ref)
    tot = (np.sum(weight) if weight is not None else len(ratio)) * M * float((amp.astype(np.float64) ** 2).sum())
    assert abs(D.sum() - tot) <= 2e-5 * tot


def test_poly_general_mask_and_limits(pyr, oracle):
    """Polychromatic plan through the general (non-separable mask) path; one wavelength at ratio 1 is the
    monochromatic plan bit for bit; bad arguments."""
    P, N, M, r, b, B = 32, 128, 6, 2.0, 2, 1
    amp, phase = inputs(P, B, 31)
    u = np.arange(N)
    f = np.where(u < N // 2, u, u - N).astype(np.float64)
    mask = (np.exp(-2j * np.pi * (N / 4) * (np.abs(f)[:, None] + np.abs(f)[None, :]) / N)
            * ((f[:, None] ** 2 + f[None, :] ** 2) <= (0.3 * N) ** 2)).astype(np.complex64)
    with pyr.Plan(P, N, M, r, b, B, poly=([1.0, 0.8], [1.0, 0.5])) as plan:
        plan.set_mask(mask)
        D, s = run(plan, amp, phase)
        with pytest.raises(pyr.PyrError):
            plan.set_double_roof(0.01)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, mask=mask.astype(np.complex128),
                                     poly=(np.float32([1.0, 0.8]).astype(np.float64), [1.0, 0.5]))
    check(D, s, D_ref, s_ref)
    with pyr.Plan(P, N, M, r, b, B, poly=([0.85], [1.5])) as plan:       # one scaled wavelength, general path
        plan.set_mask(mask)
        D, s = run(plan, amp, phase)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, mask=mask.astype(np.complex128),
                                     poly=(np.float32([0.85]).astype(np.float64), [1.5]))
    check(D, s, D_ref, s_ref)
    with pyr.Plan(P, N, M, r, b, B) as p0, pyr.Plan(P, N, M, r, b, B, poly=([1.0], None)) as p1:
        D0, s0 = run(p0, amp, phase)
        D1, s1 = run(p1, amp, phase)
    assert np.array_equal(D0, D1) and np.array_equal(s0, s1)
    for bad in [([1.0, 1.0], None), ([0.0], None), ([1.0], [-1.0])]:
        with pytest.raises(pyr.PyrError):
            pyr.Plan(P, N, M, r, b, B, poly=bad)


ROOF = [
    # P, N, M, r, b, B, kappa
    (8, 32, 4, 1.5, 1, 1, 0.01),
    (32, 128, 8, 3.0, 2, 2, 2e-3),
    (80, 256, 24, 3.0, 2, 1, -4e-4),
    (160, 512, 12, 4.0, 4, 1, 1e-4),
    (480, 2048, 4, 4.0, 8, 2, 1.5e-5),        # C5 shape (k_cols_t stages the modified y-tilt lines)
    (20, 60, 4, 2.0, 5, 1, 5e-3),             # N_fft not a power of two: table kernels
]


@pytest.mark.parametrize("P,N,M,r,b,B,kappa", ROOF)
def test_double_roof_parity(pyr, oracle, P, N, M, r, b, B, kappa):
    big = P >= 160
    amp, phase = inputs(P, B, 800 + N, sigma=2.0, eps=28 if big else 0)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        plan.set_double_roof(kappa)
        D, s = run(plan, amp, phase)
        D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, double_roof=float(np.float32(kappa)))
        check(D, s, D_ref, s_ref)
        plan.set_double_roof(0.0, enable=False)              # back to the pyramid
        D0, s0 = run(plan, amp, phase)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        D1, s1 = run(plan, amp, phase)
    assert np.array_equal(D0, D1) and np.array_equal(s0, s1)
    assert np.abs(D - D1).max() > 1e-4 * D1.max()             # the defocus between the roofs is visible


def test_half_sample_apex_mask(pyr, oracle):
    """SURVEY.md 8(f) f1 / reading S5: the apex BETWEEN four focal samples (the other common convention) is the
    separable mask g(u) = exp(-2 pi i d |f(u) + 1/2| / N); through pyr_plan_set_mask_separable, against the oracle
    with the same 2-D mask.  It differs from the on-sample apex, and a flat wavefront gives four equal pupil
    fluxes only after the half-sample tilt that centres the PSF on the shifted apex."""
    P, N, M, r, b, B = 32, 128, 8, 3.0, 2, 1
    amp, phase = inputs(P, B, 41)
    u = np.arange(N)
    f = np.where(u < N // 2, u, u - N).astype(np.float64)
    g = np.exp(-2j * np.pi * (N / 4) * np.abs(f + 0.5) / N).astype(np.complex64)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        plan.set_mask_separable(g, g)
        D, s = run(plan, amp, phase)
    mask = (g[:, None] * g[None, :]).astype(np.complex128)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, mask=mask)
    check(D, s, D_ref, s_ref)
    D_apex0, _, _ = oracle.compute(P, N, M, r, b, amp, phase)
    assert np.abs(D_ref - D_apex0).max() > 1e-3 * D_apex0.max()
    # flat wavefront + tilt of half a focal sample on both axes (phase ramp pi (x + y) / N): symmetric again
    yy, xx = np.mgrid[0:P, 0:P] - (P - 1) / 2
    ramp = (-np.pi * (xx + yy) / N).astype(np.float32)[None]
    with pyr.Plan(P, N, M, r, b, B) as plan:
        plan.set_mask_separable(g, g)
        Df, sf = run(plan, amp, ramp)
    Nq = N // b // 2
    q = [Df[0, :Nq, :Nq].sum(), Df[0, :Nq, Nq:].sum(), Df[0, Nq:, :Nq].sum(), Df[0, Nq:, Nq:].sum()]
    assert max(q) - min(q) <= 1e-4 * max(q)
