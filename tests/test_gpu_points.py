"""GPU parity for arbitrary modulation points and weights, pyr_plan_create_points (SURVEY.md 8(f) f4:
`ExtendedSource` and other modulation paths of Table 4), against the oracle's
pyr_oracle_compute_points.  Same tolerances as the circle."""
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


def random_points(M, seed, rmax=3.0, shared=True):
    rng = np.random.default_rng(seed)
    ax = rng.uniform(-rmax, rmax, M).astype(np.float32)
    ay = rng.uniform(-rmax, rmax, M).astype(np.float32)
    if shared and M >= 4:               # groups of equal y-tilt of size 3 and 2
        ay[1] = ay[0]
        ay[M - 1] = ay[0]
        ay[3] = ay[2]
    w = rng.uniform(0.0, 2.0, M).astype(np.float32)
    w[M // 2] = 0.0                     # a point that must not contribute
    return ax, ay, w


def run_and_check(pyr, oracle, P, N, b, B, pts, seed, mask=None, gx=None):
    import torch
    amp, phase = inputs(P, B, seed)
    ax, ay, w = pts
    with pyr.Plan.from_points(P, N, ax, ay, w, b, B) as plan:
        if mask is not None:
            plan.set_mask(mask)
        if gx is not None:
            plan.set_mask_separable(gx, gx)
        I, s = plan.empty_outputs()
        I.fill_(float("nan"))
        s.fill_(float("nan"))
        plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
        torch.cuda.synchronize()
        D, sl = I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)
    omask = None
    if mask is not None:
        omask = np.asarray(mask).astype(np.complex128)
    if gx is not None:
        g = np.asarray(gx).astype(np.complex128)
        omask = g[:, None] * g[None, :]
    D_ref, s_ref, _ = oracle.compute(P, N, len(ax), 0.0, b, amp, phase, mask=omask,
                                     points=(ax.astype(np.float64), ay.astype(np.float64),
                                             None if w is None else w.astype(np.float64)))
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(sl))
    dmax = np.abs(D - D_ref).max() / D_ref.max()
    l2 = np.linalg.norm((D - D_ref).ravel()) / np.linalg.norm(D_ref.ravel())
    ds = np.abs(sl - s_ref).max()
    assert dmax <= TOL_MAX and l2 <= TOL_L2 and ds <= TOL_S, "%.3e %.3e %.3e" % (dmax, l2, ds)


@pytest.mark.parametrize("P,N,M,b,B", [(8, 16, 5, 1, 1), (16, 64, 7, 2, 2), (32, 128, 9, 2, 1), (80, 256, 6, 2, 1),
                                       (120, 512, 8, 4, 2), (200, 1024, 5, 4, 1), (480, 2048, 6, 8, 1),
                                       (20, 60, 6, 5, 1)])
def test_random_points_and_weights(pyr, oracle, P, N, M, b, B):
    run_and_check(pyr, oracle, P, N, b, B, random_points(M, 40 + N), 50 + N)


def test_unit_weights_by_null(pyr, oracle):
    ax, ay, _ = random_points(6, 3)
    run_and_check(pyr, oracle, 32, 128, 2, 1, (ax, ay, None), 4)


def test_extended_source_grid(pyr, oracle):
    """An extended source: 13 x 13 points on a grid of 0.25 lambda/D with Gaussian weights (169 points,
    13 distinct y-tilts of 13 points each)."""
    g = (np.arange(13) - 6) * 0.25
    xx, yy = np.meshgrid(g, g)
    w = np.exp(-(xx ** 2 + yy ** 2) / (2 * 0.6 ** 2))
    pts = (xx.ravel().astype(np.float32), yy.ravel().astype(np.float32), w.ravel().astype(np.float32))
    run_and_check(pyr, oracle, 32, 128, 2, 1, pts, 6)


def test_points_with_general_and_separable_masks(pyr, oracle):
    N = 64
    u = np.arange(N)
    f = np.where(u < N // 2, u, u - N).astype(np.float64)
    pyramid = np.exp(-2j * np.pi * (N / 4) * (np.abs(f)[:, None] + np.abs(f)[None, :]) / N)
    stop = ((f[:, None] ** 2 + f[None, :] ** 2) <= (0.3 * N) ** 2)
    run_and_check(pyr, oracle, 16, N, 2, 1, random_points(5, 8), 9, mask=(pyramid * stop).astype(np.complex64))
    gx = np.exp(-2j * np.pi * 5 * u / N).astype(np.complex64)
    run_and_check(pyr, oracle, 16, N, 2, 1, random_points(5, 10), 11, gx=gx)


def test_circle_through_points_matches_the_circle_plan(pyr):
    import torch
    P, N, M, r, b = 32, 128, 8, 3.0, 2
    amp, phase = inputs(P, 1, 12)
    a, p = torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda()
    th = 2 * np.pi * np.arange(M) / M
    with pyr.Plan(P, N, M, r, b, 1) as p0, pyr.Plan.from_points(P, N, r * np.cos(th), r * np.sin(th), None, b, 1) as p1:
        I0, s0 = p0.empty_outputs()
        I1, s1 = p1.empty_outputs()
        p0.compute(a, p, I0, s0)
        p1.compute(a, p, I1, s1)
        torch.cuda.synchronize()
        assert (I0 - I1).abs().max().item() <= 1e-5 * I0.max().item()
        assert (s0 - s1).abs().max().item() <= 1e-5


def test_points_rejects_bad_arguments(pyr):
    with pytest.raises(pyr.PyrError):
        pyr.Plan.from_points(32, 128, np.array([0.0, np.nan], np.float32), np.zeros(2, np.float32), None, 2, 1)
    with pytest.raises(pyr.PyrError):
        pyr.Plan.from_points(32, 128, np.zeros(2, np.float32), np.zeros(2, np.float32), np.array([1.0, -1.0], np.float32), 2, 1)
