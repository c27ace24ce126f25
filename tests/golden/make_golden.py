"""Writes the stored expected values under tests/golden/ -- calls ONLY oracle/ and the seeded input recipe.

    python tests/golden/make_golden.py

yamaguchi_1S0.txt : 1S0 phase shifts (degrees) and total cross sections (mb) of the separable Yamaguchi potential
                    (reading C15; beta = 1.4488 fm^-1, a = -23.7 fm) from the oracle's MI solver (N_Q = 96,
                    PAPER.md:350 "virtually exact") at T_lab = 1, 5, 10, 25, 50, 100, 150, 200, 250, 300, 350 MeV.
                    The closed form p cot(delta) = [beta^4 - l'beta + p^2(2 beta^2 + l'/beta) + p^4]/(2 l') reproduces
                    them (tests/test_golden.py); SURVEY 8(c) C15 quotes 63.3159 / 45.8472 / 14.9765 deg at 1 / 50 / 350 MeV.
config1_1S0_N50.txt : the oracle's WPCD chain on BASELINE.json config 1 (1S0, N = 50, MT potential, 100 energies):
                    eigenvalue extremes, bound state, and every 10th phase shift -- a regression pin of the oracle itself.
No value in these files comes from the CUDA path.
"""
import math
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle as o  # noqa: E402
from paper_2106_00454_b200 import inputs as inp  # noqa: E402


def main():
    lamA, lamB = inp.yamaguchi_lambda()
    with open(os.path.join(HERE, "yamaguchi_1S0.txt"), "w") as f:
        f.write("# T_lab[MeV]  delta[deg]  sigma_tot(1S0 only)[mb]   -- oracle MI, N_Q = 96 (tests/golden/make_golden.py)\n")
        for tlab in (1.0, 5.0, 10.0, 25.0, 50.0, 100.0, 150.0, 200.0, 250.0, 300.0, 350.0):
            S, _ = o.mi_solve(tlab, kind=1, lambdaA=lamA, beta=inp.YAMAGUCHI_BETA, NQ=96)
            d = 0.5 * math.degrees(math.atan2(S.imag, S.real))
            p = math.sqrt(inp.MU * tlab) / inp.HBARC
            f.write(f"{tlab:.1f} {d:.10f} {o.sigma_tot([(0, 0, 0, 0, S)], p):.10f}\n")
    N = 50
    p = inp.grid_edges(N)
    e0, dE, Ee = o.fwp(p)
    H, V = o.assemble_H(e0, o.V_yukawa(p, 0, inp.MT_V0, inp.MT_MU))
    W, Cm, sw = o.jacobi(H)
    tl, Ecm = inp.energies(100)
    T, b = o.onshell_T(N, 0, Ee, V, W, Cm, Ecm)
    d, S = o.phase_shifts(0, T, b, dE)
    with open(os.path.join(HERE, "config1_1S0_N50.txt"), "w") as f:
        f.write("# oracle WPCD chain on config 1 (tests/golden/make_golden.py): key value(s)\n")
        f.write(f"sweeps {sw}\n")
        f.write(f"eig_min {W[0]:.12e}\neig_second {W[1]:.12e}\neig_max {W[-1]:.12e}\ntrace {W.sum():.12e}\n")
        for e in range(0, 100, 10):
            f.write(f"phase {tl[e]:.6f} {int(b[e])} {d[e]:.9f}\n")


if __name__ == "__main__":
    main()
