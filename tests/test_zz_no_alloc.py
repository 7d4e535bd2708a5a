"""The entry point that allocates nothing (`pyr_slopes_from_pixels_static`, include/pyr.h): slopes of detector frames
with the row-sum scratch in a static device array instead of plan memory, for callers that cannot call cudaMalloc.
Checked against the existing path (`pyr_slopes_from_pixels` on a plan) on two calls in a row -- the second call finds
the first call's row sums in the shared array -- and against its size limit.  Collected last on purpose (file name):
the suite runs with `pytest -x`."""
import numpy as np
import pytest

from paper_2602_06688_b200 import synth

pytestmark = pytest.mark.gpu

TOL_S = 1e-4          # north_star's slope tolerance, as in tests/test_gpu_parity.py (the two paths are in fact bit-identical)


@pytest.fixture(scope="module")
def pyr():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2602_06688_b200 import build
    build.build()
    from paper_2602_06688_b200 import pyr as m
    return m


@pytest.mark.parametrize("cfg", [1, 4, 5])
def test_static_entry_point_matches_the_plan_path_on_two_calls(pyr, cfg):
    import torch
    c = synth.CONFIGS[cfg]
    A = synth.pupil_amplitude(c.P, c.eps_pct)
    valid = synth.valid_from_amplitude(A, c.N, c.b)
    n_valid = int(valid.sum())
    Nd = c.N // c.b
    rng = np.random.default_rng(100 + cfg)
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan:
        plan.set_valid(valid)
        vd = torch.from_numpy(valid.astype(np.uint8)).cuda()
        pyr.static_scratch_init()
        for call in range(2):
            # two different frames: detector-like positive pixels, other magnitudes on the second call
            frames = torch.from_numpy(((call + 1) * 50.0 * rng.random((c.B, Nd, Nd)) + 1.0).astype(np.float32)).cuda()
            ref = torch.full((c.B, 2, Nd // 2, Nd // 2), float("nan"), device="cuda")
            got = torch.full_like(ref, float("nan"))
            plan.slopes_from_pixels(frames, ref)
            pyr.slopes_from_pixels_static(frames, vd, n_valid, got)
            torch.cuda.synchronize()
            assert torch.isfinite(got).all() and torch.isfinite(ref).all()
            assert (got - ref).abs().max().item() <= TOL_S, "call %d" % call
            assert torch.equal(got, ref), "call %d: the same kernels in the same order must agree bit for bit" % call
            assert ref.abs().max().item() > 1e-3          # the frames do have slopes


def test_static_entry_point_rejects_sizes_beyond_its_scratch(pyr):
    import torch
    Nd, B = 64, 1025                                  # 1025 * 64 = 65600 > 65536 floats of static scratch
    frames = torch.zeros((B, Nd, Nd), device="cuda")
    vd = torch.ones((Nd // 2, Nd // 2), dtype=torch.uint8, device="cuda")
    out = torch.zeros((B, 2, Nd // 2, Nd // 2), device="cuda")
    with pytest.raises(pyr.PyrError) as ei:
        pyr.slopes_from_pixels_static(frames, vd, int(vd.sum()), out)
    assert ei.value.code == 2 and "exceeds the static scratch" in str(ei.value)
    # the largest size that fits does run
    B = 1024
    frames = torch.rand((B, Nd, Nd), device="cuda") + 1.0
    out = torch.full((B, 2, Nd // 2, Nd // 2), float("nan"), device="cuda")
    pyr.slopes_from_pixels_static(frames, vd, int(vd.sum()), out)
    torch.cuda.synchronize()
    assert torch.isfinite(out).all()
