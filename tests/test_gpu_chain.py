"""GPU parity of the steps either side of the sensor (include/chain.h) against
oracle/chain_oracle.c on the same seeded inputs.

Tolerances: the CCD model and the PupData flags are integer / IEEE-exact float32 work on
both sides: bit-exact.  Atmosphere: float32 interpolation of float32 screens against double -- |d phase| <= 2e-6
(|phase| + sum_l |w_l| max|screen_l|).  Modalrec: float32 FMA sums of n terms against double -- |d modes| <= 1e-5
sum_i |R[m][i] sv[i]| (the sum of magnitudes bounds the rounding of any summation order).  Slopes from pixels:
north_star's |ds| <= 1e-4."""
import numpy as np
import pytest

from paper_2602_06688_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def chain():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2602_06688_b200 import build
    build.build()
    from paper_2602_06688_b200 import chain as m
    return m


@pytest.fixture(scope="module")
def pyr():
    from paper_2602_06688_b200 import pyr as m
    return m


@pytest.fixture(scope="module")
def oracle():
    from oracle import chain_oracle
    chain_oracle.build()
    return chain_oracle


def cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ---------------------------------------------------------------- atmosphere

def make_screens(L, S, seed):
    """Kolmogorov-like periodic screens (f^-11/6 filtered white noise on the S x S torus), float32."""
    rng = np.random.Generator(np.random.PCG64(seed))
    f = np.fft.fftfreq(S) * S
    ff = np.hypot(f[:, None], f[None, :])
    ff[0, 0] = 1.0
    filt = ff ** (-11.0 / 6.0)
    filt[0, 0] = 0.0
    out = []
    for _ in range(L):
        s = np.real(np.fft.ifft2(np.fft.fft2(rng.standard_normal((S, S))) * filt))
        out.append(s * (3.0 / s.std()))
    return np.stack(out).astype(np.float32)


@pytest.mark.parametrize("L,S,P,B", [(1, 16, 16, 1), (3, 24, 10, 2), (4, 1024, 480, 2), (4, 300, 480, 3),
                                       (20, 64, 33, 6), (16, 128, 100, 8)])
def test_atmo_parity(chain, oracle, L, S, P, B):
    import torch
    scr = make_screens(L, S, 11 + L + S)
    rng = np.random.default_rng(S)
    sh = rng.uniform(-3.0 * S, 3.0 * S, size=(B, L, 2))
    sh[0, 0] = [5.0, -7.0]                     # an integer shift
    if L > 1:
        sh[0, 1] = [0.5, 1e-9]                  # fractions at and next to the cell boundary
    w = rng.uniform(0.2, 1.5, size=L).astype(np.float32)
    with chain.Atmo(L, S, P, B, weights=w) as plan:
        out = torch.full((B, P, P), float("nan"), device="cuda")
        plan.propagate(cuda(scr), sh, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy().astype(np.float64)
    ref = oracle.atmo(scr, sh, P, weights=w.astype(np.float64))
    bound = 2e-6 * (np.abs(ref) + float((np.abs(w) * np.abs(scr).reshape(L, -1).max(1)).sum()))
    assert np.all(np.isfinite(got)) and np.all(np.abs(got - ref) <= bound), np.abs(got - ref).max()


def test_atmo_integer_shift_is_exact_and_graph_capturable(chain):
    import torch
    L, S, P, B = 1, 64, 64, 1
    scr = make_screens(L, S, 3)
    with chain.Atmo(L, S, P, B) as plan:
        out = torch.empty((B, P, P), device="cuda")
        d = cuda(scr)
        plan.propagate(d, [[[9.0, -70.0]]], out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy()[0], np.roll(scr[0], (-9, 70), axis=(0, 1)))
        st = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        out2 = torch.zeros_like(out)
        with torch.cuda.stream(st):
            plan.propagate(d, [[[1.25, 2.5]]], out2, stream=st)
            st.synchronize()
            keep = out2.clone()
            with torch.cuda.graph(g, stream=st):
                plan.propagate(d, [[[1.25, 2.5]]], out2, stream=st)
            out2.zero_()
            g.replay()
            st.synchronize()
        assert torch.equal(out2, keep)


# ---------------------------------------------------------------- CCD: bit-exact

def test_philox_stream_is_bit_exact(chain, oracle):
    import torch
    n, seed, frame = 5000, 0x0123456789ABCDEF, 77
    w = chain.philox_words(seed, frame, n)
    torch.cuda.synchronize()
    got = w.cpu().numpy().view(np.uint32)
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for i in list(range(64)) + [999, 4095, 4999]:
        assert np.array_equal(got[i], oracle.philox([i, frame, 0, 0], key)), i
    # the published known-answer vector with counter (0, 0, 0, 0), key (0, 0)
    w0 = chain.philox_words(0, 0, 1).cpu().numpy().view(np.uint32)[0]
    assert [int(v) for v in w0] == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]


CCD_CASES = [
    # shape, n_int, photon, readout, sigma, adu_gain, n_bits, gain, level
    ((1, 64, 64), 1, True, True, 0.4, 0.0, 16, 1.0, 12.0),       # Listing 2's detector: readout_level 0.4 e-
    ((2, 256, 256), 2, True, True, 1.5, 2.5, 12, 3.0, 40.0),     # both Poisson branches, ADC, clamp at 4095
    ((6, 128, 128), 3, True, False, 0.0, 0.0, 16, 0.05, 2.0),    # faint: most pixels below one electron
    ((1, 33, 47), 1, False, True, 3.0, 1.0, 8, 1.0, 100.0),      # readout noise only, 8-bit ADC
    ((2, 256, 256), 1, False, False, 0.0, 0.0, 16, 0.7, 5.0),    # noise-free: the integral itself
    ((1, 200, 200), 1, True, True, 2.0, 0.5, 30, 50.0, 4000.0),  # bright: normal branch everywhere
]


@pytest.mark.parametrize("shape,n_int,photon,readout,sigma,adu,nbits,gain,level", CCD_CASES)
def test_ccd_bit_exact(chain, oracle, shape, n_int, photon, readout, sigma, adu, nbits, gain, level):
    """Several frames, integration over n_int steps with changing intensities: the frames are identical bit for
    bit (integer draws, and float32 decisions taken with the same IEEE operations on both sides)."""
    import torch
    rng = np.random.default_rng(shape[1] + n_int)
    seed = 20260211
    ref = oracle.CCD(shape, n_int, photon, readout, sigma, adu, nbits, seed)
    with chain.CCD(shape, n_int, photon, readout, sigma, adu, nbits, seed) as ccd:
        out = torch.full(shape, float("nan"), device="cuda")
        frames = 0
        for step in range(3 * n_int + 1):
            D = (level * rng.random(shape) ** 3).astype(np.float32)     # skewed: many faint pixels, a few bright
            D[..., 0, 0] = 0.0
            r = ref.integrate(D, gain)
            ready = ccd.integrate(cuda(D), gain, out)
            torch.cuda.synchronize()
            assert ready == (r is not None)
            if ready:
                frames += 1
                got = out.cpu().numpy()
                assert np.array_equal(got, r), "frame %d: %d pixels differ" % (frames, int((got != r).sum()))
                if photon and adu == 0.0 and not readout:
                    assert np.all(got == np.rint(got)) and got.min() >= 0
        assert frames == (3 * n_int + 1) // n_int
        ccd.reset()
        ref = oracle.CCD(shape, n_int, photon, readout, sigma, adu, nbits, seed)
        D = np.full(shape, level, dtype=np.float32)
        for _ in range(n_int):
            r = ref.integrate(D, gain)
            ccd.integrate(cuda(D), gain, out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), r)      # after reset: frame 0 again, same draws


# ---------------------------------------------------------------- PupData, slopes from pixels, Modalrec

def flat_frame(pyr, c, B=1):
    """Noise-free detector frame of a flat wavefront (the calibration frame of the pupil maps)."""
    import torch
    amp = np.stack([synth.pupil_amplitude(c.P, c.eps_pct)] * B)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, B) as plan:
        I, s = plan.empty_outputs()
        plan.compute(cuda(amp), cuda(np.zeros_like(amp)), I, s)
        torch.cuda.synchronize()
        return I.cpu().numpy()


@pytest.mark.parametrize("cfg,thr", [(1, 0.3), (2, 0.3), (4, 0.25), (5, 0.3)])
def test_pupdata_bit_exact(chain, pyr, oracle, cfg, thr):
    c = synth.CONFIGS[cfg]
    ref = flat_frame(pyr, c)[0]
    v = chain.pupdata_from_frame(cuda(ref), thr)
    v0 = oracle.pupdata(ref, thr)
    assert np.array_equal(v, v0)
    geo = synth.valid_from_amplitude(synth.pupil_amplitude(c.P, c.eps_pct), c.N, c.b)
    assert abs(int(v.sum()) - int(geo.sum())) <= 0.2 * geo.sum()       # sanity: about the geometric pupil images


@pytest.mark.parametrize("cfg", [1, 3, 5])
def test_slopes_from_pixels(chain, pyr, oracle, cfg):
    """PyrSlopec on a noisy CCD frame, threshold-derived validity map: against pyro_slopes of the same frame."""
    import torch
    from oracle import pyr_oracle
    c = synth.CONFIGS[cfg]
    amp, phase = synth.make_inputs(c)
    valid = chain.pupdata_from_frame(cuda(flat_frame(pyr, c)[0]), 0.3)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan, chain.CCD((c.B, c.N_det, c.N_det), 1, True, True, 0.4, 0.0, 16, 5) as ccd:
        plan.set_valid(valid)
        I, s = plan.empty_outputs()
        plan.compute(cuda(amp), cuda(phase), I, None)
        gain = 2.0e5 / float(I[0].sum())                  # 2e5 photo-electrons per frame and source
        px = torch.empty_like(I)
        assert ccd.integrate(I, gain, px)
        s.fill_(float("nan"))
        plan.slopes_from_pixels(px, s)
        torch.cuda.synchronize()
        frames = px.cpu().numpy()
        got = s.cpu().numpy().astype(np.float64)
    for b in range(c.B):
        ref = pyr_oracle.slopes_from_D(frames[b].astype(np.float64), valid)
        assert np.abs(got[b] - ref).max() <= 1e-4
    assert np.abs(got).max() > 1e-2                     # a turbulent phase gives real slopes


@pytest.mark.parametrize("Nq,n_modes,B", [(6, 5, 1), (32, 100, 2), (64, 500, 3), (128, 1000, 2), (40, 37, 6), (20, 9, 4),
                                         (100, 70, 5), (90, 331, 1), (8, 2000, 2)])
def test_modalrec_parity(chain, oracle, Nq, n_modes, B):
    import torch
    rng = np.random.default_rng(Nq + n_modes)
    yy, xx = np.mgrid[0:Nq, 0:Nq] - (Nq - 1) / 2
    valid = ((yy ** 2 + xx ** 2 <= (0.47 * Nq) ** 2) & (yy ** 2 + xx ** 2 >= (0.13 * Nq) ** 2)).astype(np.uint8)
    nv = int(valid.sum())
    R = (rng.standard_normal((n_modes, 2 * nv)) / np.sqrt(2 * nv)).astype(np.float32)
    s = (0.3 * rng.standard_normal((B, 2, Nq, Nq))).astype(np.float32)
    s[:, :, valid == 0] = np.nan                          # invalid pixels must never be read into the product
    with chain.Modalrec(R, valid, B) as plan:
        out = torch.full((B, n_modes), float("nan"), device="cuda")
        plan.compute(cuda(s), out)
        torch.cuda.synchronize()
        got = out.cpu().numpy().astype(np.float64)
    s0 = np.nan_to_num(s)
    ref = oracle.modalrec(R, valid, s0)
    vb = valid.astype(bool)
    sv = np.concatenate([s0[:, 0][:, vb], s0[:, 1][:, vb]], axis=1).astype(np.float64)
    bound = 1e-5 * (np.abs(sv) @ np.abs(R.astype(np.float64)).T) + 1e-12
    assert np.all(np.isfinite(got)) and np.all(np.abs(got - ref) <= bound), np.abs(got - ref).max()


def test_modalrec_many_slopes_and_sources(chain, oracle):
    """20 000 slopes x 5 sources: the slope vectors of four sources do not fit shared memory next to the ring of row
    segments, so fewer sources share one pass over R (found by a random-shape sweep: the plan used to be refused)."""
    import torch
    Nq, n_modes, B = 100, 23, 5
    rng = np.random.default_rng(8)
    valid = np.ones((Nq, Nq), dtype=np.uint8)
    R = (rng.standard_normal((n_modes, 2 * Nq * Nq)) / np.sqrt(2 * Nq * Nq)).astype(np.float32)
    s = (0.3 * rng.standard_normal((B, 2, Nq, Nq))).astype(np.float32)
    with chain.Modalrec(R, valid, B) as plan:
        out = torch.full((B, n_modes), float("nan"), device="cuda")
        plan.compute(cuda(s), out)
        torch.cuda.synchronize()
        got = out.cpu().numpy().astype(np.float64)
    ref = oracle.modalrec(R, valid, s)
    sv = s.reshape(B, -1).astype(np.float64)
    bound = 1e-5 * (np.abs(sv) @ np.abs(R.astype(np.float64)).T) + 1e-12
    assert np.all(np.isfinite(got)) and np.all(np.abs(got - ref) <= bound), np.abs(got - ref).max()


def test_modalrec_identity_and_order(chain):
    import torch
    Nq = 5
    valid = np.zeros((Nq, Nq), dtype=np.uint8)
    valid[1, 2] = valid[3, 0] = valid[4, 4] = 1
    s = np.arange(2 * Nq * Nq, dtype=np.float32).reshape(1, 2, Nq, Nq)
    with chain.Modalrec(np.eye(6, dtype=np.float32), valid, 1) as plan:
        out = torch.empty((1, 6), device="cuda")
        plan.compute(cuda(s), out)
        torch.cuda.synchronize()
    assert list(out.cpu().numpy()[0]) == [7.0, 15.0, 24.0, 32.0, 40.0, 49.0]    # sx at (1,2), (3,0), (4,4), then sy


def test_modalrec_after_a_kernel_in_a_graph_and_on_a_stream(chain):
    """modalrec_compute is a programmatic dependent launch (its ring of rows of R is primed before griddepcontrol.wait):
    behind a kernel that writes the slopes -- eager on a side stream and captured in a CUDA graph -- it must see
    the finished slopes, repeat bit for bit, and be replayable."""
    import torch
    Nq, n_modes, B = 48, 700, 2
    rng = np.random.default_rng(5)
    valid = np.ones((Nq, Nq), dtype=np.uint8)
    valid[:3] = 0
    nv = int(valid.sum())
    R = (rng.standard_normal((n_modes, 2 * nv)) / np.sqrt(2 * nv)).astype(np.float32)
    base = cuda((0.3 * rng.standard_normal((B, 2, Nq, Nq))).astype(np.float32))
    with chain.Modalrec(R, valid, B) as plan:
        st = torch.cuda.Stream()
        s = torch.zeros_like(base)
        out = torch.empty((B, n_modes), device="cuda")
        with torch.cuda.stream(st):
            results = []
            for scale in (1.0, -2.0, 0.5):
                torch.mul(base, scale, out=s)          # the producer of the slopes: the kernel right before
                plan.compute(s, out, stream=st)
                results.append(out.clone())
            st.synchronize()
            ref = torch.from_numpy(R.astype(np.float64)).cuda()
            for scale, got in zip((1.0, -2.0, 0.5), results):
                sv = torch.cat([(scale * base)[:, 0][:, torch.from_numpy(valid.astype(bool)).cuda()],
                                (scale * base)[:, 1][:, torch.from_numpy(valid.astype(bool)).cuda()]], dim=1).double()
                want = sv @ ref.T
                assert (got.double() - want).abs().max().item() <= 1e-5 * (sv.abs() @ ref.abs().T).max().item()
            assert torch.equal(results[1], -2.0 * results[0])      # scaling by a power of two is exact
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                torch.mul(base, -2.0, out=s)
                plan.compute(s, out, stream=st)
            for _ in range(3):
                out.fill_(float("nan"))
                s.zero_()
                g.replay()
                st.synchronize()
                assert torch.equal(out, results[1])
