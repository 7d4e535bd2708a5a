"""GPU parity of the Shack-Hartmann path (include/sh.h) against oracle/sh_oracle.c on
the same seeded inputs.  Tolerances, derived for float32 sums of p <= 32 terms followed by F^2-term
moment sums: flux and spots 1e-5 relative (of the spot maximum for pixels),
slopes 1e-4 focal samples."""
import numpy as np
import pytest

from paper_2602_06688_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sh():
    import torch
    assert torch.cuda.is_available()
    from paper_2602_06688_b200 import build
    build.build()
    from paper_2602_06688_b200 import sh as m
    return m


@pytest.fixture(scope="module")
def oracle():
    from oracle import sh_oracle
    sh_oracle.build()
    return sh_oracle


def inputs(P, B, seed, sigma, eps=0):
    amp = np.stack([synth.pupil_amplitude(P, eps) for _ in range(B)])
    phase = np.stack([synth.kolmogorov_phase(P, amp[0], sigma, seed + s) for s in range(B)])
    return amp.astype(np.float32), phase.astype(np.float32)


def run(sh, P, n_sub, F, bs, amp, phase, spots=True):
    import torch
    with sh.Plan(P, n_sub, F, bs, amp.shape[0]) as plan:
        s, f, sp = plan.empty_outputs(spots=spots)
        s.fill_(float("nan"))
        plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), s, f, sp)
        torch.cuda.synchronize()
        return (s.cpu().numpy().astype(np.float64), f.cpu().numpy().astype(np.float64),
                None if sp is None else sp.cpu().numpy().astype(np.float64))


SHAPES = [
    # P, n_sub, F, bs, B, sigma
    (8, 2, 8, 1, 1, 1.0),
    (24, 3, 16, 2, 2, 2.0),
    (64, 8, 32, 4, 1, 3.0),
    (160, 20, 64, 4, 1, 6.0),      # 20 x 20 lenslets of 8 px, 64 x 64 samples
    (96, 3, 128, 8, 1, 8.0),       # p = 32, the largest patch
    (64, 4, 64, 4, 1, 3.0),        # p = 16: twisted radix-16 transforms
    (128, 8, 128, 8, 2, 5.0),      # p = 16, F = 128
    (40, 5, 256, 16, 2, 4.0),      # F = 256
    # the paper's own FFT sizes (Table 2): 56, 68 and 240 are not powers of two
    (160, 20, 56, 7, 1, 6.0),      # SCAO SH 314 x 56 x 56: 160 px pupil, 20 lenslets (p = 8), 8 x 8 detector pixels
    (160, 40, 68, 17, 1, 8.0),     # ERIS 1256 x 68 x 68: 40 x 40 lenslets (1256 = pi/4 40^2) of p = 4 px
    (48, 6, 240, 15, 2, 6.0),      # MORFEO FFT 240 x 240, p = 8, 16 x 16 detector pixels (full shape: test below)
    (48, 6, 240, 10, 1, 6.0),      # same, 24 x 24 pixels (three pixels per 30-column chunk)
    (32, 2, 240, 5, 1, 4.0),       # p = 16, Q = 15
    (40, 5, 56, 1, 1, 3.0),        # p = 8, no binning
    (40, 5, 56, 4, 1, 3.0),        # bs does not divide F/p: direct kernel k_sh<4,1>
    (30, 3, 68, 2, 1, 3.0),        # p = 10 (not 4/8/16), F = 68: k_sh<2,2>
    (30, 3, 240, 6, 1, 3.0),       # p = 10, F = 240: k_sh<2,2>
    (28, 2, 56, 28, 1, 3.0),       # p = 14, two pixels across: k_sh<4,1>
    # every dispatch branch of the direct kernel: RV x CU = 8x2, 4x2, 2x2, 1x2, 4x1, 2x1, 1x1, 4x4
    (20, 4, 64, 8, 1, 2.0), (20, 4, 64, 4, 1, 2.0), (20, 4, 64, 2, 1, 2.0), (20, 4, 64, 1, 1, 2.0),
    (20, 4, 32, 4, 1, 2.0), (20, 4, 32, 2, 1, 2.0), (20, 4, 32, 1, 1, 2.0),
    (20, 4, 128, 64, 1, 2.0),      # bs > 32
    (10, 2, 256, 256, 1, 2.0),     # one detector pixel per spot
]


@pytest.mark.parametrize("P,n_sub,F,bs,B,sigma", SHAPES)
def test_parity(sh, oracle, P, n_sub, F, bs, B, sigma):
    amp, phase = inputs(P, B, 900 + P + F, sigma, eps=28 if n_sub >= 8 else 0)
    s, f, sp = run(sh, P, n_sub, F, bs, amp, phase)
    s0, f0, sp0 = oracle.compute(P, n_sub, F, bs, amp, phase, want_spots=True)
    assert np.all(np.isfinite(s))
    assert np.abs(f - f0).max() <= 1e-5 * max(f0.max(), 1e-30)
    assert np.abs(sp - sp0).max() <= 1e-5 * sp0.max()
    assert np.abs(s - s0).max() <= 1e-4


def test_optional_outputs_and_determinism(sh, oracle):
    import torch
    P, n_sub, F, bs = 64, 8, 32, 2
    amp, phase = inputs(P, 2, 77, 2.0)
    s1, f1, _ = run(sh, P, n_sub, F, bs, amp, phase, spots=False)
    s2, f2, sp2 = run(sh, P, n_sub, F, bs, amp, phase, spots=True)
    assert np.array_equal(s1, s2) and np.array_equal(f1, f2)
    with sh.Plan(P, n_sub, F, bs, 2) as plan:
        s, _, _ = plan.empty_outputs()
        a, p = torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda()
        plan.compute(a, p, s)                       # flux and spots NULL
        st = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        s3 = torch.empty_like(s)
        with torch.cuda.stream(st):
            plan.compute(a, p, s3, stream=st)
            st.synchronize()
            with torch.cuda.graph(g, stream=st):
                plan.compute(a, p, s3, stream=st)
            s3.zero_()
            g.replay()
            st.synchronize()
        torch.cuda.synchronize()
        assert torch.equal(s, s3)
        assert np.array_equal(s.cpu().numpy().astype(np.float64), s1)


def test_dark_and_partial_subapertures(sh, oracle):
    P, n_sub, F, bs = 32, 4, 32, 1
    amp, phase = inputs(P, 1, 5, 1.0)
    amp[0, :8, :8] = 0.0
    amp[0, :8, 8:16] *= (np.random.default_rng(0).random((8, 8)) < 0.3)
    s, f, _ = run(sh, P, n_sub, F, bs, amp, phase, spots=False)
    s0, f0, _ = oracle.compute(P, n_sub, F, bs, amp, phase)
    assert s[0, 0, 0, 0] == 0 and s[0, 1, 0, 0] == 0 and f[0, 0, 0] == 0
    assert s[0, 0, 0, 1] == 0 and s[0, 1, 0, 1] == 0
    assert np.abs(s - s0).max() <= 1e-4 and np.abs(f - f0).max() <= 1e-5 * f0.max()


def test_morfeo_full_shape_on_a_sample(sh, oracle):
    """Table 2's largest case as the library runs it: 6 LGS x 68 x 68 lenslets (3630 = pi/4 68^2 lit), FFT 240 x 240
     -- the launch configuration bench.py times.  The oracle needs ~0.05 s per sub-aperture, so it
    is run on 3 x 3-lenslet windows of the same pupil (a sub-aperture depends on its own patch only): the pupil
    edge, the central obstruction and the interior, on three of the six sources; dark sub-apertures must be 0."""
    P, n_sub, F, bs, B, sigma = synth.SH_SHAPES["SH_MORFEO_6x3630x240x240"]
    assert (n_sub, F, B) == (68, 240, 6)
    amp, phase = synth.make_sh_inputs(P, B, sigma)
    s, f, sp = run(sh, P, n_sub, F, bs, amp, phase)
    p, w = P // n_sub, 3
    for (b, y0, x0) in [(0, 0, 32), (2, 8, 9), (5, 33, 23), (3, 40, 50), (1, 65, 30)]:
        win = (slice(b, b + 1), slice(y0 * p, (y0 + w) * p), slice(x0 * p, (x0 + w) * p))
        s0, f0, sp0 = oracle.compute(w * p, w, F, bs, amp[win], phase[win], want_spots=True)
        assert np.abs(s[b, :, y0:y0 + w, x0:x0 + w] - s0[0]).max() <= 1e-4
        assert np.abs(f[b, y0:y0 + w, x0:x0 + w] - f0[0]).max() <= 1e-5 * max(f0.max(), 1e-30)
        assert np.abs(sp[b, y0:y0 + w, x0:x0 + w] - sp0[0]).max() <= 1e-5 * max(sp0.max(), 1e-30)
    lit = (amp[0].reshape(n_sub, p, n_sub, p) ** 2).sum((1, 3))
    assert np.all(s[:, :, lit < 0.5 * p * p] == 0)
    assert abs(f.sum() - (amp.astype(np.float64) ** 2).sum()) <= 1e-5 * f.sum()      # Parseval over all sub-apertures
