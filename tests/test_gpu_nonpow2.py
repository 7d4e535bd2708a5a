"""GPU parity for N_fft that is not a power of two -- the paper's own FFT sizes are 660 (SOUL:
220 px x oversampling 3) and 1600 (ANDES: 400 px x 4).  The
library embeds the length-N circulant line operator in a power-of-two cyclic convolution; the
oracle computes the plain definition with its own mixed-radix DFT lines (pinned against the direct
O(N^2) DFT in tests/test_oracle_pins.py).  Same tolerances as everywhere.
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


def inputs(P, B, seed, sigma=1.5, eps=0):
    amp = np.stack([synth.pupil_amplitude(P, eps) for _ in range(B)])
    phase = np.stack([synth.kolmogorov_phase(P, amp[0], sigma, seed + s) for s in range(B)])
    return amp.astype(np.float32), phase.astype(np.float32)


def run_gpu(pyr, P, N, M, r, b, amp, phase, gx=None, gy=None):
    import torch
    with pyr.Plan(P, N, M, r, b, amp.shape[0]) as plan:
        if gx is not None:
            plan.set_mask_separable(gx, gy)
        I, s = plan.empty_outputs()
        I.fill_(float("nan"))
        s.fill_(float("nan"))
        plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
        torch.cuda.synchronize()
        return I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)


SHAPES = [
    # P, N, M, r, b, B
    (8, 20, 4, 1.5, 1, 1),
    (8, 24, 4, 2.0, 2, 3),
    (12, 24, 5, 1.0, 6, 1),        # P = N/2, odd M
    (20, 60, 8, 3.0, 5, 2),
    (30, 100, 5, 2.0, 5, 1),
    (44, 132, 6, 3.0, 11, 1),      # 660 / 5
    (220, 660, 24, 3.0, 5, 1),     # SOUL as Table 2 states it: 24 x 660 x 660
    (400, 1600, 24, 3.0, 8, 1),    # ANDES as Table 2 states it: 24 x 1600 x 1600; NT = 2048 embedding
    (400, 1600, 3, 4.0, 4, 2),     # same size, odd M, two sources, another binning
    # the persistent row pass (k_t2_rows) cuts the (row block, point) sequence into equal ranges: few points per
    # row block against many CTAs gives one-unit ranges (M slots of S), many sources give ranges of several row blocks
    (160, 660, 1, 2.0, 5, 1),      # one point: one unit per row block
    (160, 660, 2, 2.0, 5, 3),      # two points, three sources: two or three units per CTA
    (100, 600, 7, 2.5, 10, 2),     # odd M, ranges that start and end inside row blocks
    (300, 1200, 5, 3.0, 6, 2),     # the same at the 2048-point embedding
]


@pytest.mark.parametrize("P,N,M,r,b,B", SHAPES)
def test_parity_non_power_of_two(pyr, oracle, P, N, M, r, b, B):
    big = N >= 660
    amp, phase = inputs(P, B, 300 + N, sigma=3.0 if big else 1.5, eps=28 if big else 0)
    D, s = run_gpu(pyr, P, N, M, r, b, amp, phase)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase)
    assert np.all(np.isfinite(D)) and np.all(np.isfinite(s))
    dmax = np.abs(D - D_ref).max() / D_ref.max()
    l2 = np.linalg.norm((D - D_ref).ravel()) / np.linalg.norm(D_ref.ravel())
    ds = np.abs(s - s_ref).max()
    assert dmax <= TOL_MAX and l2 <= TOL_L2 and ds <= TOL_S, "%.3e %.3e %.3e" % (dmax, l2, ds)


def test_separable_custom_mask_non_power_of_two(pyr, oracle):
    """A pure shift mask (pin P5) at N = 60: M A^2 cyclically shifted by (dx, dy)."""
    P, N, M, r, b = 20, 60, 4, 2.0, 1
    dx, dy = 7, -4
    amp, phase = inputs(P, 1, 5)
    u = np.arange(N)
    gx = np.exp(-2j * np.pi * dx * u / N).astype(np.complex64)
    gy = np.exp(-2j * np.pi * dy * u / N).astype(np.complex64)
    D, _ = run_gpu(pyr, P, N, M, r, b, amp, phase, gx, gy)
    o = (N - P) // 2
    ref = np.zeros((N, N))
    ref[o:o + P, o:o + P] = M * amp[0].astype(np.float64) ** 2
    ref = np.roll(ref, (dy, dx), axis=(0, 1))
    assert np.abs(D[0] - ref).max() <= 1e-4 * ref.max()


def test_andes_size_properties(pyr):
    """N = 1600, P = 400 (the ANDES FFT size), beside the element-wise case above: what holds at any
    size -- Parseval (pin P3: sum D = M sum A^2) on a turbulent phase, and for
    a flat wavefront on a symmetric pupil four equal quadrant fluxes, mirror symmetry and zero
    slopes (pin P6)."""
    P, N, M, r, b = 400, 1600, 8, 3.0, 8
    amp, phase = inputs(P, 1, 77, sigma=3.0, eps=28)
    D, s = run_gpu(pyr, P, N, M, r, b, amp, phase)
    tot = M * float((amp.astype(np.float64) ** 2).sum())
    assert abs(D.sum() - tot) <= 2e-5 * tot
    D0, s0 = run_gpu(pyr, P, N, M, r, b, amp, np.zeros_like(phase))
    Nq = N // b // 2
    q = [D0[0, :Nq, :Nq].sum(), D0[0, :Nq, Nq:].sum(), D0[0, Nq:, :Nq].sum(), D0[0, Nq:, Nq:].sum()]
    assert max(q) - min(q) <= 1e-4 * max(q)
    assert np.abs(D0[0] - D0[0, ::-1, :]).max() <= 1e-4 * D0.max()
    assert np.abs(D0[0] - D0[0, :, ::-1]).max() <= 1e-4 * D0.max()
    assert np.abs(s0).max() <= 1e-4


@pytest.mark.parametrize("P,N,M,r,b,B", [(8, 20, 4, 1.5, 1, 1), (20, 60, 5, 3.0, 5, 2), (44, 132, 4, 3.0, 11, 1),
                                         (220, 660, 2, 3.0, 5, 1),       # SOUL size: the O(N^2 log N) host embedding
                                         (400, 1600, 2, 3.0, 8, 2)])     # ANDES size: embedded in 2048, the two-halves kernels k_h2_*
def test_general_mask_non_power_of_two(pyr, oracle, P, N, M, r, b, B):
    """pyr_plan_set_mask at embedded sizes: a pyramid with a field stop, and a random complex mask."""
    import torch
    u = np.arange(N)
    f = np.where(u < N // 2, u, u - N).astype(np.float64)
    pyramid = np.exp(-2j * np.pi * (N / 4) * (np.abs(f)[:, None] + np.abs(f)[None, :]) / N)
    rng = np.random.default_rng(N)
    masks = [pyramid * ((f[:, None] ** 2 + f[None, :] ** 2) <= (0.3 * N) ** 2),
             (0.5 + rng.random((N, N))) * np.exp(2j * np.pi * rng.random((N, N)))]
    amp, phase = inputs(P, B, 400 + N)
    for mask in masks:
        m32 = mask.astype(np.complex64)
        with pyr.Plan(P, N, M, r, b, B) as plan:
            plan.set_mask(m32)
            I, s = plan.empty_outputs()
            plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
            torch.cuda.synchronize()
            D, sl = I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)
        D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, mask=m32.astype(np.complex128))
        dmax = np.abs(D - D_ref).max() / D_ref.max()
        l2 = np.linalg.norm((D - D_ref).ravel()) / np.linalg.norm(D_ref.ravel())
        ds = np.abs(sl - s_ref).max()
        assert dmax <= TOL_MAX and l2 <= TOL_L2 and ds <= TOL_S, "%.3e %.3e %.3e" % (dmax, l2, ds)
