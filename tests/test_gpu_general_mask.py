"""GPU parity of the general (non-separable) focal-plane mask path, pyr_plan_set_mask, against the
CPU oracle with the same mask (field stop, other pupil separations, face
defects).  Same tolerances as the built-in path.  The oracle gets the
mask rounded to complex64 first, so input rounding is not charged to the GPU.
"""
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


def freqs(N):
    u = np.arange(N)
    return np.where(u < N // 2, u, u - N).astype(np.float64)


def mask_pyramid_sep(N, d):
    """Four-face pyramid with pupil images at +-d (d = N/4 is the built-in one)."""
    f = np.abs(freqs(N))
    return np.exp(-2j * np.pi * d * (f[:, None] + f[None, :]) / N)


def mask_field_stop(N, d, radius):
    f = freqs(N)
    stop = (f[:, None] ** 2 + f[None, :] ** 2) <= radius * radius
    return mask_pyramid_sep(N, d) * stop


def mask_defects(N, d):
    """Non-separable phase defect (a twisted face) plus a soft circular apodisation."""
    f = freqs(N)
    fu, fv = f[None, :], f[:, None]
    twist = np.exp(1j * 0.8 * np.sin(2 * np.pi * fu * fv / (N * N / 8.0)))
    apod = 1.0 / (1.0 + ((fu ** 2 + fv ** 2) / (0.35 * N) ** 2) ** 3)
    return mask_pyramid_sep(N, d) * twist * apod


def mask_zernike_dot(N, radius):
    """Zernike wavefront sensor (Table 4 `ZernikeSensor`): a pi/2 phase dot of the
    given radius (focal samples) on the optical axis, unit amplitude elsewhere."""
    f = freqs(N)
    dot = (f[:, None] ** 2 + f[None, :] ** 2) <= radius * radius
    return np.where(dot, np.exp(0.5j * np.pi), 1.0 + 0.0j)


def mask_double_roof(N, d):
    """Two crossed roof prisms in one plane would be the pyramid; a single roof splits along x only
    (`ModulatedDoubleRoof`, uses two such planes): images at +-d in x, none in y."""
    f = np.abs(freqs(N))
    return np.exp(-2j * np.pi * d * f[None, :] / N) * np.ones((N, 1))


def mask_annular_filter(N, r0, r1):
    """`FocalPlaneFilter`: a pure amplitude focal-plane mask, here an annulus."""
    f = freqs(N)
    r2 = f[:, None] ** 2 + f[None, :] ** 2
    return ((r2 >= r0 * r0) & (r2 <= r1 * r1)).astype(np.complex128)


def mask_random(N, seed):
    rng = np.random.default_rng(seed)
    return (0.5 + rng.random((N, N))) * np.exp(2j * np.pi * rng.random((N, N)))


def inputs(P, B, seed, sigma=1.5, eps=0):
    amp = np.stack([synth.pupil_amplitude(P, eps) for _ in range(B)])
    phase = np.stack([synth.kolmogorov_phase(P, amp[0], sigma, seed + s) for s in range(B)])
    return amp.astype(np.float32), phase.astype(np.float32)


def run_and_check(pyr, oracle, P, N, M, r, b, B, mask, seed, what, slopes=True):
    import torch
    amp, phase = inputs(P, B, seed)
    m32 = np.asarray(mask).astype(np.complex64)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        base = plan.launches_per_compute
        plan.set_mask(m32)
        assert plan.launches_per_compute >= base         # the three-pass general path is in use: 3 launches per chunk of points
        I, s = plan.empty_outputs()
        I.fill_(float("nan"))
        s.fill_(float("nan"))
        plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
        torch.cuda.synchronize()
        D_gpu, s_gpu = I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, mask=m32.astype(np.complex128))
    assert np.all(np.isfinite(D_gpu)) and np.all(np.isfinite(s_gpu)), what
    dmax = np.abs(D_gpu - D_ref).max() / D_ref.max()
    l2 = np.linalg.norm((D_gpu - D_ref).ravel()) / np.linalg.norm(D_ref.ravel())
    ds = np.abs(s_gpu - s_ref).max() if slopes else 0.0
    assert dmax <= TOL_MAX and l2 <= TOL_L2 and ds <= TOL_S, "%s: %.3e %.3e %.3e" % (what, dmax, l2, ds)


SHAPES = [(8, 16, 4, 1.0, 1, 1), (8, 32, 4, 1.0, 1, 1), (16, 64, 8, 2.0, 2, 2), (32, 128, 8, 3.0, 2, 1),
          (80, 256, 12, 3.0, 2, 1), (120, 512, 8, 3.0, 4, 2), (296, 1024, 4, 3.0, 4, 1)]


@pytest.mark.parametrize("P,N,M,r,b,B", SHAPES)
def test_builtin_pyramid_through_the_general_path(pyr, oracle, P, N, M, r, b, B):
    run_and_check(pyr, oracle, P, N, M, r, b, B, oracle.pyramid_mask(N), 11, "pyramid")


@pytest.mark.parametrize("P,N,M,r,b,B", SHAPES)
def test_field_stop(pyr, oracle, P, N, M, r, b, B):
    run_and_check(pyr, oracle, P, N, M, r, b, B, mask_field_stop(N, N / 4, 0.3 * N), 12, "field stop")


@pytest.mark.parametrize("P,N,M,r,b,B", SHAPES[1:6])
def test_other_separation_and_defects(pyr, oracle, P, N, M, r, b, B):
    run_and_check(pyr, oracle, P, N, M, r, b, B, mask_defects(N, N / 4 + 1.5), 13, "defects")


@pytest.mark.parametrize("P,N,M,r,b,B", SHAPES[:4])
def test_random_mask(pyr, oracle, P, N, M, r, b, B):
    run_and_check(pyr, oracle, P, N, M, r, b, B, mask_random(N, N), 14, "random mask")


@pytest.mark.parametrize("P,N,M,r,b,B", [SHAPES[3], SHAPES[5]])
def test_other_focal_plane_sensors(pyr, oracle, P, N, M, r, b, B):
    """The FFT - mask - FFT skeleton of the other sensors of Table 4: intensities of a
    Zernike phase-dot sensor, a single roof prism and an amplitude focal-plane filter (their own slope
    definitions are not part of this path, and the four-quadrant normalisation is ill-conditioned when no
    pupil image sits in the quadrants, so only the intensities are compared)."""
    run_and_check(pyr, oracle, P, N, M, r, b, B, mask_zernike_dot(N, 1.06 * N / P / 2), 21, "zernike", slopes=False)
    run_and_check(pyr, oracle, P, N, M, r, b, B, mask_double_roof(N, N / 4), 22, "roof", slopes=False)
    run_and_check(pyr, oracle, P, N, M, r, b, B, mask_annular_filter(N, 2.0, 0.35 * N), 23, "filter", slopes=False)


def test_elt_scale_chunked(pyr, oracle):
    """C5 shape (N = 2048, several chunks of modulation points), fewer points to bound the oracle time."""
    run_and_check(pyr, oracle, 480, 2048, 12, 4.0, 8, 1, mask_field_stop(2048, 512, 700.0), 15, "C5 shape")


def test_null_restores_the_previous_mask(pyr, oracle):
    import torch
    P, N, M, r, b, B = 32, 128, 8, 3.0, 2, 1
    amp, phase = inputs(P, B, 16)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        base = plan.launches_per_compute
        plan.set_mask(mask_random(N, 1).astype(np.complex64))
        assert plan.launches_per_compute > base
        plan.set_mask(None)
        assert plan.launches_per_compute == base
        I, s = plan.empty_outputs()
        plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
        torch.cuda.synchronize()
        D_gpu = I.cpu().numpy().astype(np.float64)
    D_ref, _, _ = oracle.compute(P, N, M, r, b, amp, phase)
    assert np.abs(D_gpu - D_ref).max() / D_ref.max() <= TOL_MAX


def test_general_path_is_deterministic_and_graph_capturable(pyr):
    import torch
    P, N, M, r, b, B = 32, 128, 8, 3.0, 2, 1
    amp, phase = inputs(P, B, 17)
    a, p = torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda()
    with pyr.Plan(P, N, M, r, b, B) as plan:
        plan.set_mask(mask_field_stop(N, N / 4, 40.0).astype(np.complex64))
        I1, s1 = plan.empty_outputs()
        I2, s2 = plan.empty_outputs()
        plan.compute(a, p, I1, s1)
        torch.cuda.synchronize()
        st = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(st):
            plan.compute(a, p, I2, s2)
            st.synchronize()
            with torch.cuda.graph(g, stream=st):
                plan.compute(a, p, I2, s2)
            I2.zero_()
            g.replay()
            st.synchronize()
        assert torch.equal(I1, I2) and torch.equal(s1, s2)
