"""Writes tests/golden/tiny_fx_{input,expected}.txt.  Calls ONLY the float64 oracle (oracle/), never the CUDA path.

The paper (arXiv:1801.04834) prints no worked numerical example for the correlator pipeline (SURVEY.md sec 8(c):
"the paper prints no worked example"), so this fixture is not a paper value: it freezes the oracle's own result
for a fixed tiny case (2 dual-pol stations, 16 channels, 80 int16 samples per pol, delays 0 / 1.3 us, a bandpass
ramp; readings A1-A11 of DESIGN.md) after the oracle had passed its pins, so that a later edit of the oracle's
arithmetic cannot pass unnoticed.  Regenerate only together with a commit message naming the reading that changed:

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

S, C, N = 2, 16, 80
DELAYS = np.array([0.0, 1.3e-6])
BANDPASS = 1.0 + 0.02 * np.arange(C)


def inputs():
    rng = np.random.default_rng(180104834)
    x = np.rint(rng.normal(0.0, 100.0, size=(S, 2, N, 2))).astype(np.int16)
    x[0, 0, 3] = (-32768, 32767)          # extreme values are ordinary samples (A12)
    return x


def main():
    import oracle

    x = inputs()
    vis = oracle.process_subband(x, C, DELAYS, BANDPASS, oracle.default_subband_frequency(0))
    np.savetxt(os.path.join(HERE, "tiny_fx_input.txt"), x.reshape(-1, 2), fmt="%d",
               header=f"int16 samples [S={S}][2 pol][N={N}] rows of (re, im); delays {DELAYS.tolist()} s; "
                      f"bandpass 1 + 0.02 j; subband 0 (f_sb = 100 MHz + 12 f_s)")
    np.savetxt(os.path.join(HERE, "tiny_fx_expected.txt"), vis.reshape(-1).view(np.float64).reshape(-1, 2), fmt="%.17e",
               header=f"oracle.process_subband visibilities [C={C}][n_bl=3][2][2] rows of (re, im), float64")
    print("wrote", HERE)


if __name__ == "__main__":
    main()
