"""Fixtures under tests/golden/: the paper's printed workload sizes, and an oracle-written tiny case."""
import importlib.util
import math
import os

import numpy as np
import pytest

from paper_2602_06688_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _load_maker():
    spec = importlib.util.spec_from_file_location("make_oracle_golden", os.path.join(GOLD, "make_oracle_golden.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def _stored():
    vals = np.loadtxt(os.path.join(GOLD, "oracle_tiny.txt"))
    return vals[:256].reshape(1, 16, 16), vals[256:].reshape(1, 2, 8, 8)


def test_paper_workloads_match_table2():
    rows = {}
    with open(os.path.join(GOLD, "paper_table2_workloads.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, steps, side, pupil, over = line.split()[:5]
            rows[name] = (int(steps), int(side), int(pupil), int(over))
    for key, name in (("SOUL_24x660x660", "SOUL"), ("ANDES_24x1600x1600", "ANDES")):
        c = synth.PAPER_SHAPES[key]
        steps, side, pupil, over = rows[name]
        assert (c.M, c.N, c.P) == (steps, side, pupil) and pupil * over == side
    # the flop count behind "effective FFT GFLOP/s": 2 M 2-D FFTs x 5 N^2 log2 N^2; SURVEY.md section 6
    # derives 1.96 GFLOP (SOUL) and 13.1 GFLOP (ANDES) per step from Table 2 with it
    assert abs(synth.PAPER_SHAPES["SOUL_24x660x660"].nominal_flops_per_frame / 1e9 - 1.96) < 0.01
    assert abs(synth.PAPER_SHAPES["ANDES_24x1600x1600"].nominal_flops_per_frame / 1e9 - 13.1) < 0.05
    assert math.isclose(synth.CONFIGS[5].nominal_flops_per_frame * 2, 1.181e11, rel_tol=1e-3)


def test_oracle_has_not_drifted():
    from oracle import pyr_oracle
    pyr_oracle.build()
    mk = _load_maker()
    amp, phase = mk.case_inputs()
    c = mk.CASE
    D, s, _ = pyr_oracle.compute(c["P"], c["N"], c["M"], c["r"], c["b"], amp, phase, nthreads=1)
    D0, s0 = _stored()
    assert np.allclose(D, D0, rtol=1e-12, atol=1e-14) and np.allclose(s, s0, rtol=0, atol=1e-12)


@pytest.mark.gpu
def test_gpu_against_the_stored_oracle_values():
    import torch
    from paper_2602_06688_b200 import build, pyr
    build.build()
    mk = _load_maker()
    amp, phase = mk.case_inputs()
    c = mk.CASE
    with pyr.Plan(c["P"], c["N"], c["M"], c["r"], c["b"], 1) as plan:
        I, s = plan.empty_outputs()
        plan.compute(torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda(), I, s)
        torch.cuda.synchronize()
        D, sl = I.cpu().numpy().astype(np.float64), s.cpu().numpy().astype(np.float64)
    D0, s0 = _stored()
    assert np.abs(D - D0).max() <= 1e-4 * D0.max()
    assert np.linalg.norm((D - D0).ravel()) <= 1e-5 * np.linalg.norm(D0.ravel())
    assert np.abs(sl - s0).max() <= 1e-4
