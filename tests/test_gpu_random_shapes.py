"""Seeded random shapes against the oracles: the parametrised parity tests pick their shapes by hand, this sweep does
not.  Bounded counts (about half a minute on a B200); the same loops run for minutes with other seeds found two bugs
(a polychromatic plan with one wavelength other than the reference one; a reconstructor plan whose slope vectors did
not fit shared memory four sources at a time), both fixed and pinned by cases of their own."""
import numpy as np
import pytest

from paper_2602_06688_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2602_06688_b200 import build
    build.build()
    from paper_2602_06688_b200 import pyr, sh, chain
    from oracle import pyr_oracle, sh_oracle, chain_oracle
    pyr_oracle.build()
    sh_oracle.build()
    chain_oracle.build()
    return pyr, sh, chain, pyr_oracle, sh_oracle, chain_oracle


def shape(rng, Ns, big_M=2):
    while True:
        N = int(rng.choice(Ns))
        P = int(rng.integers(1, N // 4 + 1)) * 2
        cands = [b for b in range(1, N // 4 + 1) if (N // 4) % b == 0 and (N // 4 - P // 2) % b == 0]
        if not cands:
            continue
        b = int(rng.choice(cands))
        M = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 12, 16, 24]))
        B = int(rng.choice([1, 1, 2, 3, 6]))
        if N > 256:
            M, B = min(M, big_M), min(B, 2)
        return P, N, M, float(rng.choice([0.0, 1.0, 2.5, 4.0])), b, B


def fields(P, B, seed):
    amp = np.stack([synth.pupil_amplitude(P, 0) for _ in range(B)]).astype(np.float32)
    phase = np.stack([synth.kolmogorov_phase(P, amp[0], 1.5, seed + s) for s in range(B)]).astype(np.float32)
    return amp, phase


def test_pyramid_random_shapes_masks_and_variants(mods):
    import torch
    pyr, _, _, oracle, _, _ = mods
    rng = np.random.default_rng(20260211)
    Ns = [16, 20, 24, 32, 36, 40, 48, 60, 64, 72, 96, 100, 128, 132, 160, 200, 256, 512, 660, 1024, 2048]
    for case in range(170):
        P, N, M, r, b, B = shape(rng, Ns if case % 12 == 0 else Ns[:17])
        amp, phase = fields(P, B, 9000 + case)
        mode = str(rng.choice(["builtin", "builtin", "custom", "general", "points", "poly", "roof"]))
        kw, okw = {}, {}
        u = np.arange(N)
        if mode == "points":
            ax, ay = rng.uniform(-4, 4, M).astype(np.float32), rng.uniform(-4, 4, M).astype(np.float32)
            w = rng.uniform(0.2, 2.0, M).astype(np.float32) if rng.random() < 0.6 else None
            plan = pyr.Plan.from_points(P, N, ax, ay, w, b, B)
            okw["points"] = (ax.astype(np.float64), ay.astype(np.float64), None if w is None else w.astype(np.float64))
        elif mode == "poly":
            nl = int(rng.integers(1, 4))
            ratio, wl = rng.uniform(0.7, 1.3, nl).astype(np.float32), rng.uniform(0.3, 1.5, nl).astype(np.float32)
            plan = pyr.Plan(P, N, M, r, b, B, poly=(ratio, wl))
            okw["poly"] = (ratio.astype(np.float64), wl.astype(np.float64))
        else:
            plan = pyr.Plan(P, N, M, r, b, B)
        with plan:
            if mode == "custom":
                dx, dy = int(rng.integers(-N // 2, N // 2)), int(rng.integers(-N // 2, N // 2))
                gx = np.exp(-2j * np.pi * dx * u / N).astype(np.complex64) * (1 + 0.3 * rng.random(N)).astype(np.float32)
                gy = np.exp(-2j * np.pi * dy * u / N).astype(np.complex64)
                plan.set_mask_separable(gx, gy)
                okw["mask"] = np.outer(gy, gx).astype(np.complex64)
            elif mode == "general":
                okw["mask"] = (oracle.pyramid_mask(N) * (rng.random((N, N)) > 0.2)).astype(np.complex64)
                plan.set_mask(okw["mask"])
            elif mode == "roof":
                okw["double_roof"] = float(np.float32(rng.uniform(-0.02, 0.02)))
                plan.set_double_roof(okw["double_roof"])
            I, s = plan.empty_outputs()
            I.fill_(float("nan"))
            s.fill_(float("nan"))
            plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
            torch.cuda.synchronize()
            D, sl = I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)
        D_ref, s_ref, _ = oracle.compute(P, N, M, r, b, amp, phase, **okw)
        what = "case %d %s %s" % (case, mode, (P, N, M, r, b, B))
        assert np.all(np.isfinite(D)) and np.all(np.isfinite(sl)), what
        assert np.abs(D - D_ref).max() <= 1e-4 * D_ref.max(), what
        assert np.linalg.norm((D - D_ref).ravel()) <= 1e-5 * np.linalg.norm(D_ref.ravel()), what
        if mode not in ("custom", "general"):        # (default validity map: the pupil images are where the light is)
            assert np.abs(sl - s_ref).max() <= 1e-4, what


def test_shack_hartmann_random_shapes(mods):
    import torch
    _, sh, _, _, oracle, _ = mods
    rng = np.random.default_rng(20260212)
    for case in range(70):
        p, n_sub = int(rng.integers(1, 33)), int(rng.integers(1, 6))
        P = p * n_sub
        F = max(2 * int(rng.integers(2, 65)), p + (p & 1), 4)
        if case % 9 == 0:
            F = max(int(rng.choice([56, 68, 240, 256, 500])), p + (p & 1))
        bs = int(rng.choice([d for d in range(1, F + 1) if F % d == 0]))
        B = int(rng.choice([1, 2, 3]))
        amp = (0.5 + rng.random((B, P, P))).astype(np.float32)
        phase = (1.5 * rng.standard_normal((B, P, P))).astype(np.float32)
        with sh.Plan(P, n_sub, F, bs, B) as plan:
            s, f, sp = plan.empty_outputs(spots=True)
            s.fill_(float("nan"))
            plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), s, f, sp)
            torch.cuda.synchronize()
            s, f, sp = (t.cpu().numpy().astype(np.float64) for t in (s, f, sp))
        s0, f0, sp0 = oracle.compute(P, n_sub, F, bs, amp, phase, want_spots=True)
        what = "case %d %s" % (case, (P, n_sub, F, bs, B))
        assert np.all(np.isfinite(s)) and np.abs(s - s0).max() <= 1e-4, what
        assert np.abs(f - f0).max() <= 1e-5 * f0.max() and np.abs(sp - sp0).max() <= 1e-5 * sp0.max(), what


def test_chain_random_shapes(mods):
    import torch
    _, _, chain, _, _, oracle = mods
    rng = np.random.default_rng(20260213)
    cuda = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for case in range(120):
        # CCD: bit-exact frames
        shp = (int(rng.integers(1, 4)), int(rng.integers(1, 70)), int(rng.integers(1, 70)))
        n_int, photon, ro = int(rng.integers(1, 4)), bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
        sigma, adu, nbits = float(rng.choice([0.0, 0.4, 3.0])), float(rng.choice([0.0, 0.5, 2.0])), int(rng.choice([8, 12, 16, 30]))
        seed = int(rng.integers(0, 2 ** 63))
        ref = oracle.CCD(shp, n_int, photon, ro, sigma, adu, nbits, seed)
        with chain.CCD(shp, n_int, photon, ro, sigma, adu, nbits, seed) as ccd:
            out = torch.zeros(shp, device="cuda")
            for step in range(2 * n_int + 1):
                D = (rng.random(shp) * float(rng.choice([0.01, 5.0, 40.0, 3000.0]))).astype(np.float32)
                gain = float(rng.choice([1.0, 0.37]))
                r_ = ref.integrate(D, gain)
                ready = ccd.integrate(cuda(D), gain, out)
                torch.cuda.synchronize()
                assert (r_ is not None) == ready, ("ccd", case, step)
                if ready:
                    assert np.array_equal(out.cpu().numpy(), r_), ("ccd", case, step, shp, n_int, photon, ro, sigma, adu, nbits, seed)
        # Modalrec
        Nq, nm, B = int(rng.integers(2, 100)), int(rng.integers(1, 300)), int(rng.integers(1, 7))
        valid = (rng.random((Nq, Nq)) < rng.choice([0.1, 0.6, 1.0])).astype(np.uint8)
        valid[0, 0] = 1
        nv = int(valid.sum())
        R = (rng.standard_normal((nm, 2 * nv)) / np.sqrt(2 * nv)).astype(np.float32)
        s = (0.3 * rng.standard_normal((B, 2, Nq, Nq))).astype(np.float32)
        with chain.Modalrec(R, valid, B) as plan:
            o = torch.full((B, nm), float("nan"), device="cuda")
            plan.compute(cuda(s), o)
            torch.cuda.synchronize()
            got = o.cpu().numpy().astype(np.float64)
        vb = valid.astype(bool)
        sv = np.concatenate([s[:, 0][:, vb], s[:, 1][:, vb]], axis=1).astype(np.float64)
        bound = 1e-5 * (np.abs(sv) @ np.abs(R.astype(np.float64)).T) + 1e-12
        assert np.all(np.isfinite(got)) and np.all(np.abs(got - oracle.modalrec(R, valid, s)) <= bound), ("modalrec", case, Nq, nm, B, nv)
        # atmosphere
        L, S, P, B = int(rng.integers(1, 6)), int(rng.integers(2, 200)), int(rng.integers(1, 150)), int(rng.integers(1, 4))
        scr = rng.standard_normal((L, S, S)).astype(np.float32)
        shf, w = rng.uniform(-3.0 * S, 3.0 * S, size=(B, L, 2)), rng.uniform(0.2, 1.5, size=L).astype(np.float32)
        with chain.Atmo(L, S, P, B, weights=w) as plan:
            o = torch.full((B, P, P), float("nan"), device="cuda")
            plan.propagate(cuda(scr), shf, o)
            torch.cuda.synchronize()
            got = o.cpu().numpy().astype(np.float64)
        refa = oracle.atmo(scr, shf, P, weights=w.astype(np.float64))
        bound = 2e-6 * (np.abs(refa) + float((np.abs(w) * np.abs(scr).reshape(L, -1).max(1)).sum()))
        assert np.all(np.isfinite(got)) and np.all(np.abs(got - refa) <= bound), ("atmo", case, L, S, P, B)
