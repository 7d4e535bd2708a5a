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
    (160, 20, 64, 4, 1, 6.0),      # SCAO-like: 20 x 20 lenslets of 8 px, 64 x 64 samples (Table 2: 314 x 56 x 56)
    (96, 3, 128, 8, 1, 8.0),       # p = 32, the largest patch
    (64, 4, 64, 4, 1, 3.0),        # p = 16: twisted radix-16 column transform
    (128, 8, 128, 8, 2, 5.0),      # p = 16, F = 128
    (40, 5, 256, 16, 2, 4.0),      # F = 256 (Table 2: 240 x 240)
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
