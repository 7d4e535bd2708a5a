"""Writes tests/golden/oracle_tiny.txt from the CPU oracle alone (never imports the CUDA package's
kernels: only the seeded input generator `synth`, which holds none of the method's arithmetic)."""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

CASE = dict(P=8, N=32, M=4, r=1.5, b=2, seed=20261104, sigma=1.0)


def case_inputs():
    from paper_2602_06688_b200 import synth
    A = synth.pupil_amplitude(CASE["P"], 0)
    phi = synth.kolmogorov_phase(CASE["P"], A, CASE["sigma"], CASE["seed"])
    return A[None].astype(np.float32), phi[None].astype(np.float32)


def main():
    from oracle import pyr_oracle
    pyr_oracle.build()
    amp, phase = case_inputs()
    D, s, _ = pyr_oracle.compute(CASE["P"], CASE["N"], CASE["M"], CASE["r"], CASE["b"], amp, phase, nthreads=1)
    with open(os.path.join(HERE, "oracle_tiny.txt"), "w") as f:
        f.write("# oracle/pyr_oracle.c, case %r\n" % (CASE,))
        f.write("# D [16][16] row-major, then slopes [2][8][8]; %%.17e\n")
        for v in D.ravel():
            f.write("%.17e\n" % v)
        for v in s.ravel():
            f.write("%.17e\n" % v)


if __name__ == "__main__":
    main()
