"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json:north_star's:

    max|dD| <= 1e-4 * max(D),   ||dD||_2 / ||D||_2 <= 1e-5,   max|ds| <= 1e-4.

All five BASELINE.json configs run at full size (all sources, all 16 steps of C3), in the
launch configuration bench.py times (one pyr_compute call per step on the plan's batch).
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


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(pyr, P, N, M, r, b, amp, phase, valid=None, gx=None, gy=None, want=("I", "s")):
    import torch
    B = amp.shape[0]
    with pyr.Plan(P, N, M, r, b, B) as plan:
        if valid is not None:
            plan.set_valid(valid)
        if gx is not None:
            plan.set_mask_separable(gx, gy)
        I, s = plan.empty_outputs()
        I.fill_(float("nan"))
        s.fill_(float("nan"))
        plan.compute(dev(amp), dev(phase), I if "I" in want else None, s if "s" in want else None)
        torch.cuda.synchronize()
        return I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)


def check(D_gpu, s_gpu, D_ref, s_ref, what=""):
    assert np.all(np.isfinite(D_gpu)) and np.all(np.isfinite(s_gpu)), what
    dmax = np.abs(D_gpu - D_ref).max() / D_ref.max()
    l2 = np.linalg.norm((D_gpu - D_ref).ravel()) / np.linalg.norm(D_ref.ravel())
    ds = np.abs(s_gpu - s_ref).max()
    assert dmax <= TOL_MAX, "%s max|dD|/max(D) = %.3e" % (what, dmax)
    assert l2 <= TOL_L2, "%s rel L2 = %.3e" % (what, l2)
    assert ds <= TOL_S, "%s max|ds| = %.3e" % (what, ds)
    return dmax, l2, ds


# ------------------------------------------------------------------ 1-D operator (unit level)

@pytest.mark.parametrize("N,P", [(16, 8), (32, 10), (64, 32), (128, 32), (256, 80), (512, 160),
                                 (1024, 300), (2048, 480), (2048, 1024)])
def test_line_operator_vs_oracle_1d(pyr, oracle, N, P):
    """IDFT(g . DFT(zero-pad(x)))/N per line, several CTAs plus a ragged tail of lines."""
    import torch
    rng = np.random.default_rng(N + P)
    nlines = 37
    x = (rng.normal(size=(nlines, P)) + 1j * rng.normal(size=(nlines, P))).astype(np.complex64)
    with pyr.Plan(P, N, 4, 1.0, 1, 1) as plan:
        out = plan.test_line_conv(dev(x))
        torch.cuda.synchronize()
        out = out.cpu().numpy().astype(np.complex128)
    g = oracle.pyramid_mask(N)[0, :]   # g(u) = mask[v = 0][u]
    for i in range(nlines):
        xp = np.zeros(N, complex)
        xp[:P] = x[i].astype(np.complex128)
        ref = oracle.fft1d(oracle.fft1d(xp, -1) * g, +1) / N
        err = np.abs(out[i] - ref).max() / np.abs(ref).max()
        assert err < 3e-6, "line %d: %.3e" % (i, err)


# ------------------------------------------------------------------ the five configs, full size

@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_config_parity(pyr, oracle, cfg):
    import torch
    c = synth.CONFIGS[cfg]
    A = synth.pupil_amplitude(c.P, c.eps_pct)
    valid = synth.valid_from_amplitude(A, c.N, c.b)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan:
        plan.set_valid(valid)
        assert plan.n_valid == int(valid.sum())
        I, s = plan.empty_outputs()
        for step in range(c.steps):
            amp, phase = synth.make_inputs(c, step)
            I.fill_(float("nan"))
            s.fill_(float("nan"))
            plan.compute(dev(amp), dev(phase), I, s)
            torch.cuda.synchronize()
            D_ref, s_ref, _ = oracle.compute(c.P, c.N, c.M, c.r, c.b, amp, phase, valid=valid)
            dmax, l2, ds = check(I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64),
                                 D_ref, s_ref, "C%d step %d" % (cfg, step))
            print("C%d step %d: max %.2e  L2 %.2e  slopes %.2e" % (cfg, step, dmax, l2, ds))
            # property that holds at any size: flux conservation (pin P3)
            flux = I.double().sum(dim=(1, 2)).cpu().numpy()
            assert np.allclose(flux, c.M * (amp.astype(np.float64) ** 2).sum(axis=(1, 2)), rtol=2e-5)


# ------------------------------------------------------------------ masks, maps, edge cases

def small_inputs(P, B, seed, eps_pct=0, sigma=1.5):
    A = synth.pupil_amplitude(P, eps_pct)
    amp = np.repeat(A[None], B, axis=0).copy()
    phase = np.stack([synth.kolmogorov_phase(P, A, sigma, seed + s) for s in range(B)])
    return amp, phase


def test_identity_mask_returns_the_pupil(pyr, oracle):
    """Pin P4 on the GPU: mask == 1 gives I = M |A|^2 at rows/cols o..o+P-1."""
    P, N, M, r, b = 32, 128, 8, 3.0, 1
    amp, phase = small_inputs(P, 1, 11)
    amp = amp * (1.0 + 0.5 * np.random.default_rng(3).random(amp.shape)).astype(np.float32)
    one = np.ones(N, np.complex64)
    D, _ = run_gpu(pyr, P, N, M, r, b, amp, phase, gx=one, gy=one)
    o = (N - P) // 2
    expect = np.zeros((N, N))
    expect[o:o + P, o:o + P] = M * amp[0].astype(np.float64) ** 2
    assert np.abs(D[0] - expect).max() <= 1e-4 * expect.max()


@pytest.mark.parametrize("P,N,dx,dy", [(200, 2048, 37, -411), (200, 1024, 37, -411), (300, 1024, -5, 250),
                                       (510, 1024, 401, 3), (640, 2048, 1000, -3)])
def test_separable_custom_mask_at_2048(pyr, P, N, dx, dy):
    """A custom separable mask at the two largest sizes (k_field + k_h2_cols<SEP> + k_t2_rows, one or two 1024-point
    halves per line, every pruning class): the pure shift of pin P5, I = M A^2 cyclically shifted by (dx, dy), every
    row its own line (no row twins with a custom mask)."""
    import torch
    M, r, b, B = 3, 2.0, 1, 1
    amp, phase = small_inputs(P, B, 21)
    u = np.arange(N)
    gx = np.exp(-2j * np.pi * dx * u / N).astype(np.complex64)
    gy = np.exp(-2j * np.pi * dy * u / N).astype(np.complex64)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        plan.set_mask_separable(gx, gy)
        I, s = plan.empty_outputs()
        I.fill_(float("nan"))
        plan.compute(dev(amp), dev(phase), I, s)
        torch.cuda.synchronize()
        D = I.cpu().numpy().astype(np.float64)
    o = (N - P) // 2
    ref = np.zeros((N, N))
    ref[o:o + P, o:o + P] = M * amp[0].astype(np.float64) ** 2
    ref = np.roll(ref, (dy, dx), axis=(0, 1))
    assert np.abs(D[0] - ref).max() <= 1e-4 * ref.max()


@pytest.mark.parametrize("dx,dy", [(5, 0), (0, -7), (3, 9)])
def test_shift_mask(pyr, oracle, dx, dy):
    """Pin P5 on the GPU: a pure-shift separable mask translates M |A|^2 by (+dx, +dy)."""
    P, N, M, r, b = 32, 128, 8, 3.0, 1
    amp, phase = small_inputs(P, 1, 12)
    u = np.fft.fftfreq(N) * N
    gx = np.exp(-2j * np.pi * dx * u / N).astype(np.complex64)
    gy = np.exp(-2j * np.pi * dy * u / N).astype(np.complex64)
    # every detector pixel valid: with all faces equal no light reaches the geometric pupil images, so
    # the default map would make the normalisation T rounding noise on both sides; over the whole
    # quadrant T = (total flux) / N_q^2 is well defined and the slopes of the translated pupil are compared
    valid = np.ones((N // b // 2, N // b // 2), np.uint8)
    D, s = run_gpu(pyr, P, N, M, r, b, amp, phase, valid=valid, gx=gx, gy=gy)
    o = (N - P) // 2
    base = np.zeros((N, N))
    base[o:o + P, o:o + P] = M * amp[0].astype(np.float64) ** 2
    expect = np.roll(base, (dy, dx), axis=(0, 1))
    assert np.abs(D[0] - expect).max() <= 1e-4 * expect.max()
    mask2d = gy.astype(np.complex128)[:, None] * gx.astype(np.complex128)[None, :]
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, mask=mask2d, valid=valid)
    assert np.abs(s_ref).max() > 0.1          # the comparison below is not vacuous
    check(D, s, D_ref, s_ref, "shift mask")


def test_restore_builtin_mask(pyr, oracle):
    import torch
    P, N, M, r, b = 32, 128, 8, 3.0, 2
    amp, phase = small_inputs(P, 1, 13)
    with pyr.Plan(P, N, M, r, b, 1) as plan:
        one = np.ones(N, np.complex64)
        plan.set_mask_separable(one, one)
        plan.set_mask_separable(None, None)
        I, s = plan.empty_outputs()
        plan.compute(dev(amp), dev(phase), I, s)
        torch.cuda.synchronize()
        D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase)
        check(I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64), D_ref, s_ref)


EDGE = [
    # P, N, M, r, b, B
    (2, 16, 4, 1.0, 1, 1),        # smallest sizes
    (8, 16, 4, 1.5, 4, 3),        # P = N/2 (largest pupil), b = N/4
    (16, 32, 1, 0.0, 2, 2),       # a single unmodulated point
    (16, 64, 5, 2.0, 4, 1),       # odd M (no y-tilt sharing)
    (32, 64, 6, 2.5, 1, 5),       # M even, not divisible by 4; P = N/2; ragged line groups
    (64, 128, 12, 0.0, 8, 2),     # r = 0 with M > 1 (M identical terms)
    (50, 256, 7, 3.3, 1, 3),      # P not a multiple of anything nice
    (128, 256, 8, 3.0, 64, 1),    # b = N/4: 4 x 4 detector, one pixel per quadrant ... N_q = 2
    (100, 512, 9, 5.0, 2, 2),
    (200, 1024, 8, 4.0, 4, 1),
    (512, 1024, 4, 2.0, 256, 1),  # P = N/2 at N = 1024, b = N/4
    (1024, 2048, 2, 1.0, 512, 1), # P = N/2 at the largest N
    (240, 2048, 6, 3.0, 8, 2),    # P <= N/8: the deepest pruning of the warp-per-line kernels
    (600, 2048, 3, 2.0, 4, 1),    # N/4 < P < N/2 at the largest N (no pruning), odd M
    (120, 1024, 5, 2.0, 4, 1),    # P <= N/8 at N = 1024, odd M
    (250, 2048, 3, 2.0, 1, 1),    # N_pup % 4 == 2 at the largest N: rows of R 16-byte aligned only, two-column tail block
]


@pytest.mark.parametrize("P,N,M,r,b,B", EDGE)
def test_edge_shapes(pyr, oracle, P, N, M, r, b, B):
    amp, phase = small_inputs(P, B, 100 + P + N)
    D, s = run_gpu(pyr, P, N, M, r, b, amp, phase)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase)
    check(D, s, D_ref, s_ref, str((P, N, M, r, b, B)))


def test_zero_amplitude_gives_zero_everything(pyr):
    P, N = 32, 128
    amp = np.zeros((2, P, P), np.float32)
    phase = np.ones((2, P, P), np.float32)
    D, s = run_gpu(pyr, P, N, 8, 3.0, 2, amp, phase)
    assert np.all(D == 0) and np.all(s == 0)


def test_all_invalid_map_gives_zero_slopes(pyr, oracle):
    P, N = 32, 128
    amp, phase = small_inputs(P, 1, 5)
    D, s = run_gpu(pyr, P, N, 8, 3.0, 2, amp, phase, valid=np.zeros((32, 32), np.uint8))
    assert np.all(s == 0) and D.sum() > 0


def test_large_phase_arguments(pyr, oracle):
    """|phi| up to ~60 rad: the field build must use an accurate sincos (not the fast intrinsic)."""
    P, N, M, r, b = 64, 256, 8, 3.0, 2
    amp, phase = small_inputs(P, 1, 21, sigma=15.0)
    assert np.abs(phase).max() > 30
    D, s = run_gpu(pyr, P, N, M, r, b, amp, phase)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase)
    check(D, s, D_ref, s_ref, "large phase")


def test_non_binary_amplitude_and_custom_valid(pyr, oracle):
    P, N, M, r, b = 48, 256, 12, 2.0, 4
    rng = np.random.default_rng(8)
    amp, phase = small_inputs(P, 2, 31, eps_pct=30)
    amp = (amp * rng.uniform(0.2, 2.0, size=amp.shape)).astype(np.float32)
    valid = (rng.random((N // b // 2, N // b // 2)) < 0.3).astype(np.uint8)
    D, s = run_gpu(pyr, P, N, M, r, b, amp, phase, valid=valid)
    D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, valid=valid)
    check(D, s, D_ref, s_ref, "custom valid")


def test_single_outputs(pyr, oracle):
    """Either output may be NULL; the other one is unchanged by that."""
    P, N, M, r, b = 32, 128, 8, 3.0, 2
    amp, phase = small_inputs(P, 2, 41)
    D_both, s_both = run_gpu(pyr, P, N, M, r, b, amp, phase)
    D_only, s_nan = run_gpu(pyr, P, N, M, r, b, amp, phase, want=("I",))
    D_nan, s_only = run_gpu(pyr, P, N, M, r, b, amp, phase, want=("s",))
    assert np.array_equal(D_both, D_only) and np.array_equal(s_both, s_only)
    assert np.all(np.isnan(s_nan)) and np.all(np.isnan(D_nan))   # untouched
    from paper_2602_06688_b200 import pyr as m
    with m.Plan(P, N, M, r, b, 2) as plan:
        with pytest.raises(m.PyrError) as ei:
            plan.compute(dev(amp), dev(phase), None, None)
        assert ei.value.code == m.PYR_EINVAL


def test_deterministic_and_stream_and_graph(pyr, oracle):
    """Same inputs twice -> bit-identical outputs; works on a side stream; capturable in a
    CUDA graph and replayable on new inputs (the paper's `trigger` rules)."""
    import torch
    c = synth.CONFIGS[2]
    amp, phase = synth.make_inputs(c)
    amp2, phase2 = small_inputs(c.P, c.B, 77, sigma=1.0)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan:
        a, p = dev(amp), dev(phase)
        I1, s1 = plan.empty_outputs()
        I2, s2 = plan.empty_outputs()
        plan.compute(a, p, I1, s1)
        st = torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            plan.compute(a, p, I2, s2)
        st.synchronize()
        assert torch.equal(I1, I2) and torch.equal(s1, s2)

        g = torch.cuda.CUDAGraph()
        I3, s3 = plan.empty_outputs()
        with torch.cuda.graph(g):
            plan.compute(a, p, I3, s3)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(I1, I3) and torch.equal(s1, s3)
        a.copy_(dev(amp2)); p.copy_(dev(phase2))
        g.replay()
        torch.cuda.synchronize()
        D_ref, s_ref, _ = oracle.compute(c.P, c.N, c.M, c.r, c.b, amp2, phase2)
        check(I3.cpu().numpy().astype(np.float64), s3.cpu().numpy().astype(np.float64), D_ref, s_ref, "graph replay")


def test_compute_host_matches_compute(pyr):
    import torch
    c = synth.CONFIGS[4]
    amp, phase = synth.make_inputs(c)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan:
        I, s = plan.empty_outputs()
        plan.compute(dev(amp), dev(phase), I, s)
        torch.cuda.synchronize()
        ah, ph = torch.from_numpy(amp).pin_memory(), torch.from_numpy(phase).pin_memory()
        Ih = torch.empty(I.shape, dtype=torch.float32).pin_memory()
        sh = torch.empty(s.shape, dtype=torch.float32).pin_memory()
        plan.compute_host(ah, ph, Ih, sh)
        assert torch.equal(Ih, I.cpu()) and torch.equal(sh, s.cpu())


def test_compute_host_async_pipeline(pyr):
    """pyr_compute_host_async / pyr_host_wait: six calls with different phases through the two staging slots, the
    next call enqueued before the previous one is waited for; every result equals the synchronous path bit for bit."""
    import torch
    c = synth.CONFIGS[4]
    amp, phase = synth.make_inputs(c)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan:
        I, s = plan.empty_outputs()
        phases = [np.ascontiguousarray(np.roll(phase, i, axis=2) * (1.0 + 0.1 * i)).astype(np.float32) for i in range(6)]
        refs = []
        for ph in phases:
            plan.compute(dev(amp), dev(ph), I, s)
            torch.cuda.synchronize()
            refs.append((I.cpu().clone(), s.cpu().clone()))
        ah = torch.from_numpy(amp).pin_memory()
        hp = [torch.empty(phase.shape, dtype=torch.float32).pin_memory() for _ in range(2)]
        hI = [torch.empty(I.shape, dtype=torch.float32).pin_memory() for _ in range(2)]
        hs = [torch.empty(s.shape, dtype=torch.float32).pin_memory() for _ in range(2)]
        hp[0].copy_(torch.from_numpy(phases[0]))
        plan.compute_host_async(ah, hp[0], hI[0], hs[0], slot=0)
        for i in range(1, 6):
            k = i % 2
            hp[k].copy_(torch.from_numpy(phases[i]))          # slot k was waited for two iterations ago
            plan.compute_host_async(ah, hp[k], hI[k], hs[k], slot=k)
            plan.host_wait(1 - k)
            assert torch.equal(hI[1 - k], refs[i - 1][0]) and torch.equal(hs[1 - k], refs[i - 1][1]), i
        plan.host_wait(1)
        assert torch.equal(hI[1], refs[5][0]) and torch.equal(hs[1], refs[5][1])
        plan.host_wait(0)
        with pytest.raises(pyr.PyrError):
            plan.compute_host_async(ah, hp[0], hI[0], hs[0], slot=2)


@pytest.mark.parametrize("P,N,M,r,b,B,jc", [(480, 2048, 12, 4.0, 8, 2, 0), (480, 2048, 7, 3.0, 8, 1, 1), (250, 2048, 6, 2.0, 1, 1, 2),
                                            (600, 2048, 5, 2.0, 4, 2, 2)])
def test_l2_resident_schedule(pyr, oracle, P, N, M, r, b, B, jc):
    """pyr_plan_set_schedule: the two passes per chunk of y-tilts with R as a two-chunk ring (several ring wraps, a
    ragged last chunk, odd M, chunk of one y-tilt): same tolerances against the oracle; switching back restores the
    single-pass result bit for bit; other sizes refuse."""
    import torch
    amp, phase = small_inputs(P, B, 77 + M)
    with pyr.Plan(P, N, M, r, b, B) as plan:
        I, s = plan.empty_outputs()
        plan.compute(dev(amp), dev(phase), I, s)
        torch.cuda.synchronize()
        I0, s0 = I.clone(), s.clone()
        base = plan.launches_per_compute
        plan.set_schedule(True, jc)
        assert plan.launches_per_compute > base
        I.fill_(float("nan")); s.fill_(float("nan"))
        for _ in range(2):                                   # second call: the ring is reused
            plan.compute(dev(amp), dev(phase), I, s)
        torch.cuda.synchronize()
        D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase)
        check(I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64), D_ref, s_ref, "chunked")
        plan.set_schedule(False)
        plan.compute(dev(amp), dev(phase), I, s)
        torch.cuda.synchronize()
        assert torch.equal(I, I0) and torch.equal(s, s0)
    with pyr.Plan(32, 128, 8, 3.0, 2, 1) as plan:
        with pytest.raises(pyr.PyrError):
            plan.set_schedule(True)


def test_binding_rejects_wrong_tensors(pyr):
    import torch
    with pyr.Plan(32, 128, 8, 3.0, 2, 1) as plan:
        I, s = plan.empty_outputs()
        good = torch.zeros((1, 32, 32), device="cuda")
        with pytest.raises(TypeError):
            plan.compute(good.cpu(), good, I, s)
        with pytest.raises(TypeError):
            plan.compute(good.double(), good, I, s)
        with pytest.raises(ValueError):
            plan.compute(torch.zeros((1, 32, 31), device="cuda"), good, I, s)
        with pytest.raises(TypeError):
            plan.compute(good, torch.zeros((1, 32, 64), device="cuda")[:, :, ::2], I, s)
