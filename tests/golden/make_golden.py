"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ and the seeded input
generators -- never the CUDA path.  Run from the repo root:  python tests/golden/make_golden.py

  c0_transmission.txt : T_LR(E) and ||X||_F per energy of BASELINE.json config 0 (oracle/dense.py, Tier A).
  impurity_chain.txt  : textbook closed form T = (2 t sin k)^2 / ((2 t sin k)^2 + V^2) of a 1-D chain with one
                        impurity (t = -1, V = 0.7, site 5 of 9), evaluated from the formula, not from any solver.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import dense  # noqa: E402
from paper_1812_01396_b200 import inputs  # noqa: E402


def main():
    p = inputs.make_problem(inputs.CONFIGS["C0"])
    X, T = dense.solve_all(p)
    with open(os.path.join(HERE, "c0_transmission.txt"), "w") as f:
        f.write("# BASELINE.json config 0 (bs=16 nb=8 seed 0), oracle/dense.py; columns: Re E, Im E, T_LR, ||X||_F\n")
        for e in range(p.n_energy):
            f.write(f"{p.E[e].real:.17e} {p.E[e].imag:.17e} {T[e]:.17e} {np.linalg.norm(X[e]):.17e}\n")
    t, V = -1.0, 0.7
    E = inputs.energy_grid(7, -1.9, 1.9, 0.0).real
    k = np.arccos(E / (2 * t))
    v2 = (2 * t * np.sin(k)) ** 2
    with open(os.path.join(HERE, "impurity_chain.txt"), "w") as f:
        f.write("# closed form, 1-D chain t=-1 with one impurity V=0.7: columns: E, T(E)\n")
        for a, b in zip(E, v2 / (v2 + V * V)):
            f.write(f"{a:.17e} {b:.17e}\n")


if __name__ == "__main__":
    main()
