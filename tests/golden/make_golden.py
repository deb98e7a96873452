"""Writes tests/golden/wilson_clover_2x4x2x4.txt.  Calls ONLY wdinputs/ and oracle/ (never the CUDA path).

The paper prints no worked numerical example, so this fixture is not a paper value: it is the
pinned oracle's own output (eq. 1.13) on a tiny seeded case, stored so that a
later change of the oracle's arithmetic or of the input generators shows up as a diff.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import wdinputs  # noqa: E402

DIMS, M0, CSW, SEED_U, EPS, SEED_PSI = (2, 4, 2, 4), -0.4, 1.0, 7001, 0.4, 7002
SAMPLES = [(0, 0), (1, 5), (17, 11), (30, 3), (42, 7), (63, 0), (63, 11), (21, 9)]


def compute():
    U = wdinputs.gauge_exp(DIMS, SEED_U, EPS)
    psi = wdinputs.spinor(DIMS, SEED_PSI)[0]
    C = oracle.build_clover(DIMS, M0, CSW, U)
    return U, psi, C, oracle.apply(DIMS, M0, U, C, psi), oracle.apply(DIMS, M0, U, None, psi)


if __name__ == "__main__":
    U, psi, C, out_c, out_w = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "wilson_clover_2x4x2x4.txt")
    with open(path, "w") as fh:
        fh.write("# oracle output of eq. 1.13 (PAPER.md:227-230); written by tests/golden/make_golden.py\n")
        fh.write(f"# dims={DIMS} m0={M0} csw={CSW} gauge=exp(i*{EPS}*H) seed {SEED_U}, spinor seed {SEED_PSI}\n")
        fh.write("# kind site component re im\n")
        for s, k in SAMPLES:
            fh.write(f"clover {s} {k} {out_c[s, k, 0]:.17g} {out_c[s, k, 1]:.17g}\n")
        for s, k in SAMPLES:
            fh.write(f"wilson {s} {k} {out_w[s, k, 0]:.17g} {out_w[s, k, 1]:.17g}\n")
        fh.write(f"norm2_clover -1 -1 {float((out_c ** 2).sum()):.17g} 0\n")
        fh.write(f"norm2_wilson -1 -1 {float((out_w ** 2).sum()):.17g} 0\n")
        fh.write(f"norm2_input -1 -1 {float((psi ** 2).sum()):.17g} 0\n")
    print("wrote", path)
